"""paper_1111_0716_b200 — plane-wave Fock exchange (V_x|psi>, E_x) on one B200, hand-written sm_100a CUDA.

`workloads` (seeded inputs) imports without the CUDA library; everything else lives in `binding` and fails
loudly when libexx.so is missing.
"""
