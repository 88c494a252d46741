"""amrhydro: B200-native batched finite-volume update for block-structured AMR patches.

Hot path of Wang, Abel & Kaehler (arXiv:0910.5547): TVD-RK2 / PLM / HLL(LLF) per-patch
update plus CFL reduction, ghost fill, restriction and refluxing, as sm_100a CUDA kernels
behind the C ABI declared in include/amrhydro.h.  `workloads` holds the seeded inputs;
`binding` is the thin ctypes layer over libamrhydro.so (argument marshalling only).
"""
