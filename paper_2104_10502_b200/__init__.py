"""B200-native H|psi> (plane-wave pseudopotential Kohn-Sham Hamiltonian application).

`inputs` (seeded workload generators) imports without the CUDA extension; the binding (`qe_hpsi`) loads
`libqe_hpsi.so` lazily and fails loudly when it is missing -- there is no CPU fallback.
"""
