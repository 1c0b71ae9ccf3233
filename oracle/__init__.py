"""CPU oracle for the Wilson-Dirac / Neuberger-Dirac hot path of arXiv:1010.5636.

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only `tests/`, `__graft_entry__.smoke()` and the
`cpu_baseline` / `--impl reference` legs of `bench.py` may import or execute anything under `oracle/`.
The CUDA path (`paper_1010_5636_b200/`) never imports it and shares no code, header, table or
constant with it; both read only the seeded input generators in `lattice_inputs/`.

Everything here is plain fp64 numpy (plus one plain-C restatement of eq. 2.1, `wilson_ref.c`, used
where numpy is too slow) written from the paper's equations in the paper's notation: full 4x4 gamma
matrices, full 3x3 links, no spin-projection shortcut, no link compression inside the operator, no
blocking or fusion.  Every function cites the passage it follows; every reading of a point where the
paper is silent is listed in DESIGN.md section 3.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): point source written out by hand from eq. 2.1,
Hermiticity, free-field plane-wave closed form, gauge covariance, literal site-loop brute force, dense
4^4 eigendecomposition -> exact sign(Q), Ginsparg-Wilson relation, scalar polynomial bound delta,
compression round trips.  No function in this package is "parity unpinned".
"""
