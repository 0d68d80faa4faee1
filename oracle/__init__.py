"""fp64 CPU oracle of the NEP3 hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports paper_2205_10046_b200 and shares no code with the CUDA library.
"""
from .nep_oracle import (  # noqa: F401
    OracleHyper, build, lib, num_threads, num_descriptors, fc, fk, bk, bk_grad, constants, q_from_S,
    ann, neighbors, neighbors_of, compute, md, latent, heat_current, kinetic_temperature, md_berendsen,
    ACC_CONV, KB_EV_PER_K, counter_normal, langevin_half_step, md_langevin, loss_terms, regularisation_terms,
    compute_images, count_images, loss_terms_batch, last_timing,
)
