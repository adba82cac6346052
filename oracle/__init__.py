"""CPU oracle for the BatchTNMC hot path (arXiv 2509.19006) -- TEST INFRASTRUCTURE ONLY.

Plain, slow, FP64 numpy restatement of what the hot path computes, written from
/root/reference/PAPER.md (cited as PAPER.md:NN) and the readings listed in DESIGN.md.
It shares no code with the CUDA path (`paper_2509_19006_b200/`): neither imports the
other.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import anything from here; the product path never does.

Modules
-------
exact       E1 energy (Eq. 1), E2 brute-force Z / Boltzmann / conditionals (Eq. 2-4),
            E3 exact row-transfer-matrix state vectors (Fig. 1b restated)
bmps        C0-C3 boundary-MPS cache build: Boltzmann matrices (Eq. 7), copy tensors
            (Eq. 8), bottom row, row MPO, MPO x MPS, compress (reading P-C2), log Z
sampler     S1-S2 right-environment sweep and left sampling sweep
metropolis  S4 independence Metropolis scan (Eq. 10)
observables thermal averages of E and M along the accepted chain (reading G19)
philox      Part R counter-based uniforms, Philox4x32-10, indexed (disorder, sample, site)

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): closed forms, brute force on <=4x4,
exact-chi limit, ferromagnetic limit, Eckart-Young, sum_s q(s) = 1, gauge covariance,
cuRAND's header implementation of Philox4x32-10 and the Random123 known-answer vectors.
"parity unpinned" items: the sweep order / truncation convention of
`compress` (P-C2) cannot be compared with the paper's own code, which is not available.
"""
