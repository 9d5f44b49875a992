"""Pins of the oracle's mixed-precision defect correction (oracle/hz_oracle.py, reading R27; PAPER.md:229
"Since the DDM is a preconditioner, we can gain significant speedups simply by evaluating the preconditioner in
a lower precision").  CPU only.

Expected values come from the already pinned plain iteration (`ddm_sweep`, an exact algebraic identity links
the two) and from the sparse direct solve of the global system; nothing is produced by the function under test.
"""
import numpy as np

from oracle import hz_oracle as O
from paper_2606_21695_b200.inputs import make_config


def problem_from(inp):
    return O.Problem(inp.nx, inp.ny, inp.p, inp.x0, inp.y0, inp.x1, inp.y1, inp.c_nodes, inp.omega,
                     inp.f_re.astype(complex))


def rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def test_a_cycle_without_rounding_is_m_plain_sweeps():
    # X + sum_{j<m} T^j (F(X) - X) = F^m(X) for the affine sweep map F = T . + c: exact identity, so a dropped
    # term, a homogeneous sweep that still carries the load, or an off-by-one in m shows at 1e-12.
    rng = np.random.default_rng(3)
    shape = (4 * 2 + 1, 6 * 2 + 1)
    bc = [rng.standard_normal(n) + 1j * rng.standard_normal(n) for n in (shape[0], shape[0], shape[1], shape[1])]
    pr = O.Problem(6, 4, 2, 0.0, 0.0, 1.5, 0.8, 1.0 + rng.uniform(0, 1.5, size=shape), 9.0,
                   (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)), bc)
    for m, cycles in ((1, 3), (4, 2), (7, 1)):
        st = O.ddm_setup(pr, 3, 2, 0.5)
        pr0 = O.Problem(pr.nx, pr.ny, pr.p, pr.x0, pr.y0, pr.x1, pr.y1, pr.c_nodes, pr.omega, np.zeros_like(pr.f))
        st_h = O.ddm_setup(pr0, 3, 2, 0.5, n_t=st.tab.n_t)
        for _ in range(cycles):
            O.ddm_mixed_cycle(st, st_h, m, 2, 0.5, lo_dtype=None)
        ref = O.ddm_solve(pr, 3, 2, m * cycles, 2, True, 0.5)
        assert rel(O.ddm_pack(st), O.ddm_pack(ref)) < 1e-12, (m, cycles)


def test_float32_correction_converges_to_the_direct_solve_where_a_float32_state_stalls():
    # config 1 (2x2 subdomains, p=2): the fp64-accumulated iteration with the correction stored in float32
    # reaches the direct solve <= 1e-8 (north_star's bar for the converged DDM) ...
    inp = make_config(1)
    pr = problem_from(inp)
    ustar = O.direct_solve(pr)
    st = O.ddm_mixed_solve(pr, inp.sx, inp.sy, 40, 10, 2, 0.5, lo_dtype=np.complex64)
    err_mixed = rel(O.ddm_gather(st), ustar)
    assert err_mixed < 1e-8, err_mixed
    assert O.residual(pr, O.ddm_gather(st)) < 1e-7
    # ... whereas the same number of plain sweeps with the STATE itself stored in float32 stalls two orders
    # of magnitude above it (the rounding error is then relative to |X|, not to the correction)
    st32 = O.ddm_setup(pr, inp.sx, inp.sy, 0.5)
    for _ in range(400):
        O.ddm_sweep(st32, 2, True, 0.5)
        O._state_round(st32, np.complex64)
    err_plain = rel(O.ddm_gather(st32), ustar)
    assert err_plain > 30 * err_mixed, (err_plain, err_mixed)
    # and the rounded cycles track the unrounded ones (i.e. the plain fp64 iteration) to float32 accuracy
    a = O.ddm_mixed_solve(pr, inp.sx, inp.sy, 3, 10, 2, 0.5, lo_dtype=np.complex64)
    b = O.ddm_solve(pr, inp.sx, inp.sy, 30, 2, True, 0.5)
    assert rel(O.ddm_pack(a), O.ddm_pack(b)) < 1e-5
