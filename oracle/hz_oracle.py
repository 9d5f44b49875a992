"""CPU ORACLE for the block-level DDM / WaveHoltz hot path of arxiv/paper_2606_21695.

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, fp64 numpy/scipy
restatement of what the paper computes, written from /root/reference/PAPER.md only.
Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import it.  It shares no code, table or constant
generator with `paper_2606_21695_b200/` (the CUDA path) and never imports it.

Citations are "PAPER.md:<line> (section / equation)".  Where the paper is silent,
garbled or inconsistent the reading is the one listed in DESIGN.md ("Readings", R1..R24).

What is pinned (tests/test_oracle_pins.py; none of the pins re-types a formula below):
  gll()                      sum(w)=2, D exact on polynomials, symmetry, Lambda_1=4, Lambda_2=24
  element_stiffness()        A_e 1 = 0, symmetric, exact energy of a polynomial field
  assemble_global()/direct   plane wave recovered at order ~h^(2p) (eq. (1))
  wh_tables()                filter orthogonality identities
  waveholtz_iteration()      fixed point == dense direct solve of (4),
                             leapfrog evolves e^{-i w t} exactly at every step
  ddm_*()                    converged DDM == dense direct solve <=1e-8,
                             L=1 DDM == WaveHoltz on the whole domain, hand-sized 2x1 case,
                             wrong sign of eq. (2) diverges (reading R3)
  ddm_gmres()                (tests/test_oracle_gmres_pins.py) iterate == least-squares minimiser over an
                             explicitly built Krylov basis (numpy lstsq, tiny case), converged == dense direct
                             solve, monotone residuals, sweep map affine / real-linear
  ddm_mixed_cycle()/_solve() (tests/test_oracle_mixed_pins.py) without rounding a cycle == m plain sweeps (exact
                             identity), with the correction stored in float32 it still converges to the dense direct
                             solve <= 1e-8 where the plain iteration with a float32 state stalls above it
  minres()/block_system()    (tests/test_oracle_minres_pins.py) symmetry/indefiniteness of (5), iterate == residual
                             minimiser over an explicit Krylov basis, recurrence residual == true residual,
                             converged == dense direct solve, agreement with scipy.sparse.linalg.minres
  quad_geometry()/element_stiffness_quad()/region_operators_quads()/choose_nt_quads()
                             (tests/test_oracle_quads_pins.py) rectangles reduce to the pinned rectangular operators,
                             patch test (A x linear = 0 inside), exact area / first moment / side lengths, the
                             N_t bound really bounds lmax(M^-1 A), plane wave recovered at high order on a
                             distorted mesh, converged DDM == direct solve on a distorted mesh
Nothing here is "parity unpinned".

Conventions
  mesh      nx*ny rectangular elements on [x0,x1]x[y0,y1], degree p, GLL nodes;
            global node (I,J), I in 0..nx*p, J in 0..ny*p, flat index J*(nx*p+1)+I (x fastest).
  sides     0=W (I=0), 1=E (I=max), 2=S (J=0), 3=N (J=max); an edge array runs along
            increasing J (W,E) or increasing I (S,N) and INCLUDES both end nodes.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as spla

W_, E_, S_, N_ = 0, 1, 2, 3
OPPOSITE = (E_, W_, N_, S_)


# --------------------------------------------------------------------------------------
# O1  Discretisation: GLL nodal basis (Section IV)
# --------------------------------------------------------------------------------------
def gll(p: int):
    """Gauss-Lobatto-Legendre nodes xi_0..xi_p on [-1,1] (roots of (1-x^2) P_p'(x)),
    weights w_a = 2 / (p (p+1) P_p(xi_a)^2) and the Lagrange differentiation matrix
    D[a,b] = l_b'(xi_a).  PAPER.md:113 ("GLL quadrature rule on which the nodal basis is
    defined"), PAPER.md:199 ("1D differentiation matrix D of size (P+1)^2")."""
    if p < 1:
        raise ValueError("p >= 1")
    Pp = np.polynomial.legendre.Legendre.basis(p)
    interior = np.sort(np.real(Pp.deriv().roots())) if p > 1 else np.array([])
    xi = np.concatenate(([-1.0], interior, [1.0]))
    # polish the interior roots with Newton on P_p'(x)
    d1, d2 = Pp.deriv(), Pp.deriv(2)
    for _ in range(4):
        if p > 1:
            xi[1:-1] -= d1(xi[1:-1]) / d2(xi[1:-1])
    w = 2.0 / (p * (p + 1) * Pp(xi) ** 2)
    D = np.zeros((p + 1, p + 1))
    # barycentric form of the derivative of the Lagrange basis
    bw = np.array([1.0 / np.prod([xi[a] - xi[b] for b in range(p + 1) if b != a])
                   for a in range(p + 1)])
    for a in range(p + 1):
        for b in range(p + 1):
            if a != b:
                D[a, b] = (bw[b] / bw[a]) / (xi[a] - xi[b])
        D[a, a] = -np.sum(D[a, :])
    return xi, w, D


def stiffness_1d(p: int):
    """Reference 1-D stiffness K = D^T W D on [-1,1] (A_ij=(grad phi_j, grad phi_i)
    with GLL quadrature, evaluated through D as in PAPER.md:201)."""
    _, w, D = gll(p)
    return D.T @ np.diag(w) @ D


def lambda_p(p: int) -> float:
    """Largest eigenvalue of the 1-D element pencil (K_h, W_h) at element length h=1
    (reading R9: it bounds the spectrum of M^-1 A and fixes the stable time step)."""
    _, w, _ = gll(p)
    K = stiffness_1d(p)
    # physical element of length h: K_h = (2/h) K, W_h = (h/2) W  ->  W_h^-1 K_h = (2/h)^2 W^-1 K
    ev = np.linalg.eigvals(np.diag(1.0 / w) @ K)
    return float(4.0 * np.max(np.real(ev)))


def element_stiffness(p: int, hx: float, hy: float):
    """(p+1)^2 x (p+1)^2 stiffness of one hx-by-hy rectangle, local node (a,b) -> b*(p+1)+a.
    int grad(phi_j).grad(phi_i) with GLL quadrature: (hy/hx) W(x)K  [d/dx part]
    + (hx/hy) K(x)W [d/dy part]; np.kron(Y, X)[b*(p+1)+a, ...] = Y[b,.] X[a,.].
    PAPER.md:109 (definition of A), PAPER.md:199-201 (gradient via D, then D^T)."""
    _, w, _ = gll(p)
    K = stiffness_1d(p)
    Wm = np.diag(w)
    return (hy / hx) * np.kron(Wm, K) + (hx / hy) * np.kron(K, Wm)


# --------------------------------------------------------------------------------------
# Problem description (eq. (1); arguments mirror include/hz.h)
# --------------------------------------------------------------------------------------
@dataclass
class Problem:
    nx: int
    ny: int
    p: int
    x0: float
    y0: float
    x1: float
    y1: float
    c_nodes: np.ndarray          # (ny*p+1, nx*p+1) wave speed AT the global GLL nodes (R14)
    omega: float
    f: np.ndarray                # (ny*p+1, nx*p+1) complex source AT the nodes
    bc_lambda: list | None = None  # 4 complex edge arrays (W,E,S,N) or None (=0)
    vx: np.ndarray | None = None   # F3: (ny+1, nx+1) vertex coordinates of straight-sided convex quads on a
    vy: np.ndarray | None = None   #     logically rectangular mesh; when given, x0..y1 are ignored

    @property
    def hx(self):
        return (self.x1 - self.x0) / self.nx

    @property
    def hy(self):
        return (self.y1 - self.y0) / self.ny

    @property
    def npx(self):
        return self.nx * self.p + 1

    @property
    def npy(self):
        return self.ny * self.p + 1

    def node_coords(self):
        xi, _, _ = gll(self.p)
        x = np.concatenate([self.x0 + self.hx * (e + (xi[:-1] + 1) / 2) for e in range(self.nx)]
                           + [[self.x1]])
        y = np.concatenate([self.y0 + self.hy * (e + (xi[:-1] + 1) / 2) for e in range(self.ny)]
                           + [[self.y1]])
        return x, y


def _region_operators(p, ex, ey, hx, hy):
    """Assemble, by summation over the ex*ey elements of a rectangular region, the
    stiffness A (sparse), the geometric lumped mass m (one value per region node) and the
    geometric edge weights s[side] (one value per edge node) of that region.
    PAPER.md:109-113: GLL quadrature makes M and H diagonal.  Lumped mass of element node
    (a,b): (hx/2)(hy/2) w_a w_b; edge weight of an element-edge node: (h_edge/2) w_a."""
    _, w, _ = gll(p)
    Ae = element_stiffness(p, hx, hy)
    npx, npy = ex * p + 1, ey * p + 1
    rows, cols, vals = [], [], []
    m = np.zeros((npy, npx))
    la = np.arange(p + 1)
    for fy in range(ey):
        for fx in range(ex):
            gi = (fy * p + la)[:, None] * npx + (fx * p + la)[None, :]   # [b,a] -> global
            gi = gi.reshape(-1)
            rows.append(np.repeat(gi, (p + 1) ** 2))
            cols.append(np.tile(gi, (p + 1) ** 2))
            vals.append(Ae.reshape(-1))
            m[fy * p:fy * p + p + 1, fx * p:fx * p + p + 1] += (hx / 2) * (hy / 2) * np.outer(w, w)
    A = sp.csr_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))),
                      shape=(npx * npy, npx * npy))
    A.sum_duplicates()
    sy = np.zeros(npy)
    for fy in range(ey):
        sy[fy * p:fy * p + p + 1] += (hy / 2) * w
    sx = np.zeros(npx)
    for fx in range(ex):
        sx[fx * p:fx * p + p + 1] += (hx / 2) * w
    s = [sy.copy(), sy.copy(), sx.copy(), sx.copy()]
    return A, m, s


def edge_index(npx, npy, side):
    """Flat region indices of the nodes of one side, in the edge-array order."""
    if side == W_:
        return np.arange(npy) * npx
    if side == E_:
        return np.arange(npy) * npx + (npx - 1)
    if side == S_:
        return np.arange(npx)
    return (npy - 1) * npx + np.arange(npx)


# --------------------------------------------------------------------------------------
# O2  Global reference system (4) and direct solve (eq. (4))
# --------------------------------------------------------------------------------------
def assemble_global(pr: Problem):
    """Returns A (sparse real), M (diag, real), H (diag, real; outer boundary only), b (complex)
    of  (A - i w H - w^2 M) u = b,  PAPER.md:105-111."""
    if pr.vx is not None:
        A, m, s = region_operators_quads(pr.p, pr.vx, pr.vy)
    else:
        A, m, s = _region_operators(pr.p, pr.nx, pr.ny, pr.hx, pr.hy)
    c = np.asarray(pr.c_nodes, dtype=float).reshape(-1)
    M = m.reshape(-1) / c ** 2
    H = np.zeros_like(M)
    b = np.asarray(pr.f, dtype=complex).reshape(-1) * m.reshape(-1)
    for side in range(4):
        idx = edge_index(pr.npx, pr.npy, side)
        H[idx] += s[side] / c[idx]
        if pr.bc_lambda is not None:
            b[idx] += s[side] * np.asarray(pr.bc_lambda[side], dtype=complex)
    return A, M, H, b


def helmholtz_matrix(A, M, H, omega):
    return (A.astype(complex) - sp.diags(1j * omega * H + omega ** 2 * M)).tocsc()


def direct_solve(pr: Problem):
    """Sparse LU of the global discrete Helmholtz system (4): the plain definition of the
    converged answer."""
    A, M, H, b = assemble_global(pr)
    u = spla.splu(helmholtz_matrix(A, M, H, pr.omega)).solve(b)
    return u.reshape(pr.npy, pr.npx)


def residual(pr: Problem, u):
    """|| b - (A - i w H - w^2 M) u ||_2 / || b ||_2 on the global system (row A10 of the scope
    table; the operator is the paper's "Operator time" normaliser)."""
    A, M, H, b = assemble_global(pr)
    u = np.asarray(u, dtype=complex).reshape(-1)
    r = b - (A @ u - (1j * pr.omega * H + pr.omega ** 2 * M) * u)
    return float(np.linalg.norm(r) / np.linalg.norm(b))


# --------------------------------------------------------------------------------------
# O4  WaveHoltz (Section V; Algorithm 1 at PAPER.md:160-183)
# --------------------------------------------------------------------------------------
def choose_nt(p, hx, hy, c_max, omega, cfl_frac):
    """Number of time steps per period T = 2 pi / w (reading R9).  The stable step of the
    leapfrog is dt_stab = 2 / sqrt(lmax) with lmax = c_max^2 Lambda_p (1/hx^2 + 1/hy^2) the
    bound on the spectrum of M^-1 A; N_t = ceil(T / (cfl_frac dt_stab)), at least 4.  The
    paper prints only dt <= 2h/(p^2 c_max), which is not a bound in 2-D."""
    lmax = c_max ** 2 * lambda_p(p) * (1.0 / hx ** 2 + 1.0 / hy ** 2)
    dt_stab = 2.0 / math.sqrt(lmax)
    T = 2.0 * math.pi / omega
    return max(4, int(math.ceil(T / (cfl_frac * dt_stab) * (1.0 - 1e-12))))


@dataclass
class WHTables:
    n_t: int
    dt: float
    theta: float
    sigma: float
    kappa: np.ndarray        # kappa_nu,       nu = 0..N_t-1
    kappa_half: np.ndarray   # kappa_{nu+1/2}, nu = 0..N_t-1
    cos_nu: np.ndarray       # cos(2 pi nu / N_t)
    sin_nu: np.ndarray       # sin(2 pi nu / N_t)


def wh_tables(n_t: int, omega: float) -> WHTables:
    """Filter kappa_nu = cos(2 pi nu/N_t) - 1/4 + 1/4 tan^2(pi/N_t), evaluated at
    nu and at nu+1/2 (reading R6); theta = tan(w dt/2)/w, sigma = sin(w dt/2)/(w/2)
    (PAPER.md:144)."""
    dt = 2.0 * math.pi / omega / n_t
    nu = np.arange(n_t, dtype=float)

    def kap(x):
        return np.cos(2 * np.pi * x / n_t) - 0.25 + 0.25 * math.tan(math.pi / n_t) ** 2

    return WHTables(n_t=n_t, dt=dt,
                    theta=math.tan(omega * dt / 2) / omega,
                    sigma=math.sin(omega * dt / 2) / (omega / 2),
                    kappa=kap(nu), kappa_half=kap(nu + 0.5),
                    cos_nu=np.cos(2 * np.pi * nu / n_t), sin_nu=np.sin(2 * np.pi * nu / n_t))


def waveholtz_iteration(A, M, H, b, u, omega, tab: WHTables, trace=None):
    """One application of Pi (eq. (7)) in the order of Algorithm 1
    (PAPER.md:168-178).  A sparse real, M/H real diagonals, b/u complex vectors.
    If `trace` is a list, (p^nu, pdot^{nu+1/2}) of every step is appended to it."""
    N = tab.n_t
    alpha = (M - tab.theta * H) / (M + tab.theta * H)
    beta = tab.sigma / (M + tab.theta * H)
    # Initialise p <- Re u ; pdot <- Re{-i w u e^{-pi i / N_t}}  (reading R8)
    p = np.real(u).copy()
    pdot = np.real(-1j * omega * u * np.exp(-1j * math.pi / N))
    # v <- kappa_0 p - (1/(i w)) kappa_{1/2} pdot   (eq. (7) sign, reading R2)
    v = tab.kappa[0] * p - (1.0 / (1j * omega)) * tab.kappa_half[0] * pdot
    if trace is not None:
        trace.append((p.copy(), pdot.copy()))
    for nu in range(1, N):                                     # PAPER.md:170 (reading R5)
        p = p + tab.sigma * pdot                               # PAPER.md:142 / 172
        Ap = A @ p
        src = np.real(b * np.exp(-2j * math.pi * nu / N))      # PAPER.md:140 (reading R7)
        pdot = alpha * pdot + beta * (-Ap + src)               # PAPER.md:140 / 176
        v = v + tab.kappa[nu] * p - (1.0 / (1j * omega)) * tab.kappa_half[nu] * pdot  # 177
        if trace is not None:
            trace.append((p.copy(), pdot.copy()))
    return (2.0 / N) * v                                       # eq. (7) prefactor (reading R4)


# --------------------------------------------------------------------------------------
# O3/O5/O6/O7  Domain decomposition (Section III; Algorithm 1)
# --------------------------------------------------------------------------------------
@dataclass
class Subdomain:
    ix: int                      # position in the sx*sy subdomain grid
    iy: int
    I0: int                      # global node offset of the local node (0,0)
    J0: int
    npx: int
    npy: int
    A: sp.csr_matrix             # local stiffness (own elements only)
    M: np.ndarray                # c^-2 * local lumped mass
    H: np.ndarray                # c^-1 * edge weight on the WHOLE subdomain boundary (O3)
    bf: np.ndarray               # f(x_j) * local lumped mass (+ physical-side bc_lambda), complex
    s: list                      # geometric edge weights per side
    k_edge: list                 # k_j = omega / c_j on each side's nodes (reading R15)
    neighbour: list              # subdomain index across each side, or -1 (physical boundary)
    edge_idx: list = field(default_factory=list)


@dataclass
class DDMState:
    pr: Problem
    sx: int
    sy: int
    tab: WHTables
    subs: list
    lam: list                    # lam[l][side] complex edge array (zeros on physical sides)
    u: list                      # u[l] complex local vector (previous WaveHoltz iterate)
    n_sweeps: int = 0


def split_elements(n: int, s: int):
    """Sizes and offsets of the s consecutive groups n elements are split into (reading R25): floor(n/s) each,
    the first n mod s groups one more."""
    q, r = divmod(n, s)
    sizes = [q + 1 if k < r else q for k in range(s)]
    offs = [k * q + min(k, r) for k in range(s)]
    return sizes, offs


def ddm_setup(pr: Problem, sx: int, sy: int, cfl_frac: float = 0.5, n_t: int | None = None) -> DDMState:
    """Partition into sx*sy rectangular subdomains of about (nx/sx)*(ny/sy) elements and build the
    subdomain systems (O3): A_l, M_l from the subdomain's own elements; H_l on its whole
    boundary (interfaces carry the same impedance operator as the outer boundary,
    PAPER.md:70-75, 83); load f(x_j) m^l_j with the LOCAL mass."""
    if not (1 <= sx <= pr.nx and 1 <= sy <= pr.ny):
        raise ValueError("need 1 <= sx <= nx, 1 <= sy <= ny")
    # Ragged partitions (reading R25; "at most K elements", fn. at 203): the nx element columns are
    # split as evenly as possible, the first nx mod sx subdomain columns get one element more; same in y.
    exs, X0 = split_elements(pr.nx, sx)
    eys, Y0 = split_elements(pr.ny, sy)
    quads = pr.vx is not None
    c = np.asarray(pr.c_nodes, dtype=float)
    f = np.asarray(pr.f, dtype=complex)
    if n_t is None:
        if quads:
            n_t = choose_nt_quads(pr.p, pr.vx, pr.vy, c, pr.omega, cfl_frac)
        else:
            n_t = choose_nt(pr.p, pr.hx, pr.hy, float(c.max()), pr.omega, cfl_frac)
    tab = wh_tables(n_t, pr.omega)
    subs = []
    rect_ops = {}
    for iy in range(sy):
        for ix in range(sx):
            ex, ey = exs[ix], eys[iy]
            npx, npy = ex * pr.p + 1, ey * pr.p + 1
            I0, J0 = X0[ix] * pr.p, Y0[iy] * pr.p
            if quads:   # F3: the subdomain's own elements, from its block of the vertex arrays
                A, m, s = region_operators_quads(pr.p, pr.vx[Y0[iy]:Y0[iy] + ey + 1, X0[ix]:X0[ix] + ex + 1],
                                                 pr.vy[Y0[iy]:Y0[iy] + ey + 1, X0[ix]:X0[ix] + ex + 1])
            else:
                if (ex, ey) not in rect_ops:
                    rect_ops[(ex, ey)] = _region_operators(pr.p, ex, ey, pr.hx, pr.hy)
                A, m, s = rect_ops[(ex, ey)]
            cl = c[J0:J0 + npy, I0:I0 + npx].reshape(-1)
            fl = f[J0:J0 + npy, I0:I0 + npx].reshape(-1)
            M = m.reshape(-1) / cl ** 2
            H = np.zeros_like(M)
            bf = fl * m.reshape(-1)
            nb = [-1, -1, -1, -1]
            if ix > 0:
                nb[W_] = iy * sx + ix - 1
            if ix < sx - 1:
                nb[E_] = iy * sx + ix + 1
            if iy > 0:
                nb[S_] = (iy - 1) * sx + ix
            if iy < sy - 1:
                nb[N_] = (iy + 1) * sx + ix
            eidx, kedge = [], []
            for side in range(4):
                idx = edge_index(npx, npy, side)
                eidx.append(idx)
                H[idx] += s[side] / cl[idx]
                kedge.append(pr.omega / cl[idx])
                if nb[side] < 0 and pr.bc_lambda is not None:
                    full = np.asarray(pr.bc_lambda[side], dtype=complex)
                    off = J0 if side in (W_, E_) else I0
                    bf[idx] += s[side] * full[off:off + len(idx)]
            subs.append(Subdomain(ix, iy, I0, J0, npx, npy, A, M, H, bf, s, kedge, nb, eidx))
    lam = [[np.zeros(len(sd.edge_idx[side]), dtype=complex) for side in range(4)] for sd in subs]
    u = [np.zeros(sd.npx * sd.npy, dtype=complex) for sd in subs]
    return DDMState(pr, sx, sy, tab, subs, lam, u)


def ddm_cycle(st: DDMState, l: int, n_wh: int, warm_start: bool, sign_2ik: float = -1.0):
    """Algorithm 1 on subdomain l.  Returns (u_l, g) where g[side] is the
    outgoing interface datum of each non-physical side (None on physical sides):
        g = -lambda^n_{l,side} - 2 i k u_l      (eq. (2), sign per reading R3;
    `sign_2ik=+1` reproduces the printed sign and is used only by the pin that shows it
    diverges)."""
    sd = st.subs[l]
    # Assemble b from f and lambda^n: b_j = f_j m_j + sum_sides s_j lambda_j
    b = sd.bf.copy()
    for side in range(4):
        if sd.neighbour[side] >= 0:
            b[sd.edge_idx[side]] += sd.s[side] * st.lam[l][side]
    # u^(0) <- 0 or the previous iterate (warm start, reading R11)
    u = st.u[l].copy() if warm_start else np.zeros_like(st.u[l])
    for _ in range(n_wh):                                   # fixed count (reading R10)
        u = waveholtz_iteration(sd.A, sd.M, sd.H, b, u, st.pr.omega, st.tab)
    g = [None] * 4
    for side in range(4):
        if sd.neighbour[side] >= 0:
            g[side] = -st.lam[l][side] + sign_2ik * 2j * sd.k_edge[side] * u[sd.edge_idx[side]]
    return u, g


def ddm_sweep(st: DDMState, n_wh: int, warm_start: bool, relax: float, sign_2ik: float = -1.0):
    """One outer iteration: the DDM cycle on every subdomain from the SAME lambda^n (all
    subdomains concurrently), then the exchange (O6): subdomain l's outgoing g
    on `side` lands in neighbour r's slot on the opposite side, with relaxation rho (R12):
        lambda^{n+1}_{r,opp} = (1-rho) lambda^n_{r,opp} + rho g_{l,side}."""
    L = len(st.subs)
    new_u, gs = [None] * L, [None] * L
    for l in range(L):
        new_u[l], gs[l] = ddm_cycle(st, l, n_wh, warm_start, sign_2ik)
    new_lam = [[a.copy() for a in st.lam[l]] for l in range(L)]
    for l in range(L):
        for side in range(4):
            r = st.subs[l].neighbour[side]
            if r >= 0:
                o = OPPOSITE[side]
                new_lam[r][o] = (1.0 - relax) * st.lam[r][o] + relax * gs[l][side]
    st.lam, st.u = new_lam, new_u
    st.n_sweeps += 1
    return st


def ddm_gather(st: DDMState):
    """Global nodal field: mean of the copies at nodes shared by several subdomains (R19)."""
    pr = st.pr
    acc = np.zeros((pr.npy, pr.npx), dtype=complex)
    cnt = np.zeros((pr.npy, pr.npx))
    for l, sd in enumerate(st.subs):
        acc[sd.J0:sd.J0 + sd.npy, sd.I0:sd.I0 + sd.npx] += st.u[l].reshape(sd.npy, sd.npx)
        cnt[sd.J0:sd.J0 + sd.npy, sd.I0:sd.I0 + sd.npx] += 1.0
    return acc / cnt


def ddm_solve(pr: Problem, sx: int, sy: int, n_outer: int, n_wh: int, warm_start: bool = True,
              relax: float = 0.5, cfl_frac: float = 0.5, n_t: int | None = None,
              sign_2ik: float = -1.0, state: DDMState | None = None):
    """n_outer sweeps from lambda^0 = 0, u^0 = 0 (or continue `state`)."""
    st = state if state is not None else ddm_setup(pr, sx, sy, cfl_frac, n_t)
    for _ in range(n_outer):
        ddm_sweep(st, n_wh, warm_start, relax, sign_2ik)
    return st


# --------------------------------------------------------------------------------------
# R27  Mixed-precision outer iteration ("Since the DDM is a preconditioner, we can gain
#      significant speedups simply by evaluating the preconditioner in a lower precision")
# --------------------------------------------------------------------------------------
# One warm-started sweep is an affine map F(X) = T X + c of the joint state X = (lambda, u_l) (see F2 below);
# T is the same sweep with the load removed (f = 0, boundary datum = 0).  Defect correction in that state
# space, X kept in fp64:
#     D        = F(X) - X                          one sweep at full precision
#     delta_1  = lo(D)
#     delta_k+1 = lo(T delta_k + D),  k = 1..m-1   m-1 homogeneous sweeps whose state is stored at LOW precision
#     X       <- X + delta_m
# Without rounding (lo = identity) delta_m = sum_{j<m} T^j D and X + delta_m = F^m(X) exactly: the cycle IS m
# plain sweeps.  With rounding the low-precision sweeps only ever see the correction, so their rounding error
# is relative to |delta|, not to |X|, and the fixed point is still that of the full-precision map (D = 0).
def _state_copy(st: DDMState):
    return [[a.copy() for a in sides] for sides in st.lam], [a.copy() for a in st.u]


def _state_round(st: DDMState, lo_dtype) -> None:
    if lo_dtype is None:
        return
    st.lam = [[a.astype(lo_dtype).astype(complex) for a in sides] for sides in st.lam]
    st.u = [a.astype(lo_dtype).astype(complex) for a in st.u]


def ddm_mixed_cycle(st: DDMState, st_h: DDMState, m_inner: int, n_wh: int, relax: float, lo_dtype=np.complex64):
    """One defect-correction cycle on `st` (state X, load f).  `st_h` is a DDMState of the SAME problem with
    f = 0 and no boundary datum (the homogeneous sweep T); its state is scratch."""
    lam0, u0 = _state_copy(st)
    ddm_sweep(st, n_wh, True, relax)                                   # F(X), full precision
    Dl = [[a - b for a, b in zip(sa, sb)] for sa, sb in zip(st.lam, lam0)]
    Du = [a - b for a, b in zip(st.u, u0)]
    st_h.lam, st_h.u = [[a.copy() for a in sides] for sides in Dl], [a.copy() for a in Du]
    _state_round(st_h, lo_dtype)                                       # delta_1 = lo(D)
    for _ in range(m_inner - 1):
        ddm_sweep(st_h, n_wh, True, relax)                             # T delta_k
        st_h.lam = [[a + d for a, d in zip(sa, sd)] for sa, sd in zip(st_h.lam, Dl)]
        st_h.u = [a + d for a, d in zip(st_h.u, Du)]
        _state_round(st_h, lo_dtype)
    st.lam = [[a + d for a, d in zip(sa, sd)] for sa, sd in zip(lam0, st_h.lam)]
    st.u = [a + d for a, d in zip(u0, st_h.u)]
    return st


def ddm_mixed_solve(pr: Problem, sx: int, sy: int, n_cycles: int, m_inner: int, n_wh: int, relax: float = 0.5,
                    cfl_frac: float = 0.5, lo_dtype=np.complex64):
    """n_cycles defect-correction cycles from X = 0.  Returns the fp64 state."""
    st = ddm_setup(pr, sx, sy, cfl_frac)
    pr0 = Problem(pr.nx, pr.ny, pr.p, pr.x0, pr.y0, pr.x1, pr.y1, pr.c_nodes, pr.omega,
                  np.zeros_like(pr.f), None, vx=pr.vx, vy=pr.vy)
    st_h = ddm_setup(pr0, sx, sy, cfl_frac, n_t=st.tab.n_t)
    for _ in range(n_cycles):
        ddm_mixed_cycle(st, st_h, m_inner, n_wh, relax, lo_dtype)
    return st


# --------------------------------------------------------------------------------------
# F2  Krylov acceleration of the outer iteration (the fixed-point iteration on
#     lambda "can be accelerated with a Krylov space method")
# --------------------------------------------------------------------------------------
# One warm-started sweep is an affine map x -> F(x) = T x + c of the joint state
# x = (lambda on all interface sides, u_l of all subdomains); its fixed point is the DDM fixed
# point (u_l = exact subdomain solutions, lambda consistent), i.e. the global discrete solution.
# T is only REAL-linear (WaveHoltz takes real parts), so x is packed as a real
# vector (real parts, then imaginary parts) with the Euclidean inner product.
# Restarted GMRES(m) on (I - T) x = c: Arnoldi with modified Gram-Schmidt, least-squares problem
# by Givens rotations (Saad & Schultz 1986, in its textbook form).  Each Arnoldi step costs one sweep.
def ddm_pack(st: DDMState, with_u: bool = True) -> np.ndarray:
    parts = []
    for l, sd in enumerate(st.subs):
        for side in range(4):
            if sd.neighbour[side] >= 0:
                parts.append(st.lam[l][side])
    if with_u:
        parts += st.u
    z = np.concatenate(parts)
    return np.concatenate([z.real, z.imag])


def ddm_unpack(st: DDMState, x: np.ndarray, with_u: bool = True) -> None:
    h = len(x) // 2
    z = x[:h] + 1j * x[h:]
    o = 0
    for l, sd in enumerate(st.subs):
        for side in range(4):
            if sd.neighbour[side] >= 0:
                n = len(st.lam[l][side])
                st.lam[l][side] = z[o:o + n].copy()
                o += n
    if not with_u:
        return
    for l in range(len(st.subs)):
        n = len(st.u[l])
        st.u[l] = z[o:o + n].copy()
        o += n


# Krylov iteration on lambda ALONE (the fixed-point iteration on the interface data "accelerated with a
# Krylov space method").  With a COLD start (Algorithm 1 as printed, u^(0) = 0) and a
# fixed number n_wh of WaveHoltz iterations, one sweep is an affine, real-linear map lambda -> G lambda + d of the
# interface data alone (u_l is an output, not a state), so GMRES on (I - G) lambda = d needs basis vectors of the size of
# the interfaces only.  Its fixed point is the DDM fixed point of the INEXACT subdomain solver (n_wh WaveHoltz iterations
# from zero); it tends to the discrete solution as n_wh grows.  After the iteration the field is u_l(lambda) by one more
# cycle at fixed lambda, optionally polished by `n_polish` further warm-started WaveHoltz iterations at that lambda.
def ddm_gmres(pr: Problem, sx: int, sy: int, n_wh: int, relax: float, restart: int, n_steps: int,
              cfl_frac: float = 0.5, tol: float = 0.0, lambda_only: bool = False, n_polish: int = 0):
    """Runs `n_steps` Arnoldi steps in total (restarting every `restart` steps) of GMRES on
    (I - T) x = c from x = 0 and leaves the final iterate in the returned state.
    Returns (state, history) with history[k] = relative LINEAR residual ||c - (I-T)x_k|| / ||c||
    after k steps, as estimated by the Givens recurrence.  Stops early when that drops to `tol`.
    lambda_only: x = lambda and the sweeps are cold-started (see above); the returned state then holds
    u_l = n_wh (+ n_polish warm-started) WaveHoltz iterations for the final lambda."""
    st = ddm_setup(pr, sx, sy, cfl_frac)
    with_u = not lambda_only

    def F(x):
        ddm_unpack(st, x, with_u)
        ddm_sweep(st, n_wh, with_u, relax)
        return ddm_pack(st, with_u)

    x = np.zeros_like(ddm_pack(st, with_u))
    c = F(x)
    cnorm = float(np.linalg.norm(c))
    hist = [1.0]
    done = 0
    while done < n_steps and cnorm > 0:
        r = c - (x - (F(x) - c)) if done > 0 else c.copy()
        beta = float(np.linalg.norm(r))
        m = min(restart, n_steps - done)
        V = [r / beta]
        H = np.zeros((m + 1, m))
        cs, sn = np.zeros(m), np.zeros(m)
        g = np.zeros(m + 1)
        g[0] = beta
        k = 0
        for j in range(m):
            w = V[j] - (F(V[j]) - c)                       # (I - T) v_j
            for i in range(j + 1):                          # modified Gram-Schmidt
                H[i, j] = float(V[i] @ w)
                w = w - H[i, j] * V[i]
            H[j + 1, j] = float(np.linalg.norm(w))
            V.append(w / H[j + 1, j])
            for i in range(j):                              # previous rotations on the new column
                t = cs[i] * H[i, j] + sn[i] * H[i + 1, j]
                H[i + 1, j] = -sn[i] * H[i, j] + cs[i] * H[i + 1, j]
                H[i, j] = t
            d = math.hypot(H[j, j], H[j + 1, j])
            cs[j], sn[j] = H[j, j] / d, H[j + 1, j] / d
            H[j, j], H[j + 1, j] = d, 0.0
            g[j + 1] = -sn[j] * g[j]
            g[j] = cs[j] * g[j]
            k = j + 1
            done += 1
            hist.append(abs(g[j + 1]) / cnorm)
            if tol > 0 and hist[-1] <= tol:
                break
        y = np.linalg.solve(np.triu(H[:k, :k]), g[:k])
        for i in range(k):
            x = x + y[i] * V[i]
        if tol > 0 and hist[-1] <= tol:
            break
    ddm_unpack(st, x, with_u)
    if lambda_only:                                         # u_l(lambda) at the final lambda (lambda itself is not advanced)
        for l in range(len(st.subs)):
            st.u[l], _ = ddm_cycle(st, l, n_wh, False)
        if n_polish > 0:
            for l in range(len(st.subs)):
                st.u[l], _ = ddm_cycle(st, l, n_polish, True)
    return st, hist


# --------------------------------------------------------------------------------------
# F1  MINRES as the subdomain solver: the paper's comparator (eq. (5), 123, 271-277)
# --------------------------------------------------------------------------------------
def block_system(A, M, H, b, omega):
    """The real symmetric indefinite 2N x 2N form (5) of (4):
        [[A - w^2 M, w H], [w H, w^2 M - A]] [Re u; Im u] = [Re b; -Im b]."""
    D = sp.diags(omega ** 2 * M)
    Hm = sp.diags(omega * H)
    K = sp.bmat([[A - D, Hm], [Hm, D - A]]).tocsr()
    rhs = np.concatenate([np.real(b), -np.imag(b)])
    return K, rhs


def minres(K, rhs, x0=None, tol=1e-12, max_iters=10000, history=None):
    """MINRES of Paige & Saunders (1975) in its textbook Lanczos / Givens form, no preconditioner, for the
    symmetric indefinite system K x = rhs ("five vectors and two inner products per iteration",
    PAPER.md:123, 275).  Stops when the recurrence's residual norm |eta| <= tol * ||rhs|| (the relative
    residual the paper iterates to: 1e-6 in single, 1e-12 in double precision).
    Returns (x, iterations)."""
    n = len(rhs)
    x = np.zeros(n) if x0 is None else np.array(x0, dtype=float)
    bnorm = float(np.linalg.norm(rhs))
    v = rhs - K @ x
    gamma = float(np.linalg.norm(v))            # gamma_1
    if history is not None:
        history.append(gamma / bnorm if bnorm > 0 else 0.0)
    if bnorm == 0.0 or gamma <= tol * bnorm:
        return x, 0
    eta = gamma
    v_old = np.zeros(n)
    w_old, w = np.zeros(n), np.zeros(n)         # w_{j-1}, w_j
    s_old, s, c_old, c = 0.0, 0.0, 1.0, 1.0
    it = 0
    for it in range(1, max_iters + 1):
        v = v / gamma
        Kv = K @ v
        delta = float(v @ Kv)
        v_new = Kv - delta * v - gamma * v_old
        gamma_new = float(np.linalg.norm(v_new))
        a0 = c * delta - c_old * s * gamma
        a1 = math.hypot(a0, gamma_new)
        a2 = s * delta + c_old * c * gamma
        a3 = s_old * gamma
        c_new, s_new = a0 / a1, gamma_new / a1
        w_new = (v - a3 * w_old - a2 * w) / a1
        x = x + c_new * eta * w_new
        eta = -s_new * eta
        if history is not None:
            history.append(abs(eta) / bnorm)
        v_old, v, gamma = v, v_new, gamma_new
        w_old, w = w, w_new
        s_old, s, c_old, c = s, s_new, c, c_new
        if abs(eta) <= tol * bnorm or gamma == 0.0:
            break
    return x, it


def ddm_cycle_minres(st: DDMState, l: int, tol: float, max_iters: int, warm_start: bool):
    """The DDM cycle of Algorithm 1 with MINRES on (5) in place of the WaveHoltz loop.
    Returns (u_l, g, iterations)."""
    sd = st.subs[l]
    b = sd.bf.copy()
    for side in range(4):
        if sd.neighbour[side] >= 0:
            b[sd.edge_idx[side]] += sd.s[side] * st.lam[l][side]
    K, rhs = block_system(sd.A, sd.M, sd.H, b, st.pr.omega)
    x0 = np.concatenate([st.u[l].real, st.u[l].imag]) if warm_start else None
    x, its = minres(K, rhs, x0, tol, max_iters)
    n = len(b)
    u = x[:n] + 1j * x[n:]
    g = [None] * 4
    for side in range(4):
        if sd.neighbour[side] >= 0:
            g[side] = -st.lam[l][side] - 2j * sd.k_edge[side] * u[sd.edge_idx[side]]
    return u, g, its


def ddm_sweep_minres(st: DDMState, tol: float, max_iters: int, warm_start: bool, relax: float):
    """One outer iteration with MINRES subdomain solves; returns the iteration counts."""
    L = len(st.subs)
    new_u, gs, its = [None] * L, [None] * L, [0] * L
    for l in range(L):
        new_u[l], gs[l], its[l] = ddm_cycle_minres(st, l, tol, max_iters, warm_start)
    new_lam = [[a.copy() for a in st.lam[l]] for l in range(L)]
    for l in range(L):
        for side in range(4):
            r = st.subs[l].neighbour[side]
            if r >= 0:
                o = OPPOSITE[side]
                new_lam[r][o] = (1.0 - relax) * st.lam[r][o] + relax * gs[l][side]
    st.lam, st.u = new_lam, new_u
    st.n_sweeps += 1
    return its


# --------------------------------------------------------------------------------------
# F3  General straight-sided convex quadrilaterals ("quadrilateral ... elements",
#     gradient through D, "geometric factors" at the quadrature points, then D^T;
#     SURVEY.md section 8(f) F3).  The mesh is logically rectangular: element (fx,fy) has the vertices
#     (vx,vy)[fy:fy+2, fx:fx+2]; each element is the bilinear image of the reference square [-1,1]^2.
#     Pins: tests/test_oracle_quads_pins.py (rectangles reduce to _region_operators, patch test,
#     exact area / first moment / side lengths, plane-wave convergence on a distorted mesh,
#     converged DDM == direct solve on a distorted mesh).
# --------------------------------------------------------------------------------------
def quad_geometry(p: int, X4, Y4):
    """Element map x(xi,eta) = sum_k N_k(xi,eta) x_k with the bilinear N_k; X4[b][a] is the vertex at
    (xi,eta) = (2a-1, 2b-1).  Returns, at the (p+1)^2 GLL points [b,a] (eta index first):
    x, y, detJ and the three geometric factors of  grad u . grad v detJ = (u_xi,u_eta) g (v_xi,v_eta)^T,
    g = detJ J^-1 J^-T  (J = d(x,y)/d(xi,eta)):  gxx = (x_eta^2+y_eta^2)/detJ,
    gxy = -(x_xi x_eta + y_xi y_eta)/detJ, gyy = (x_xi^2+y_xi^2)/detJ."""
    xi, _, _ = gll(p)
    X4, Y4 = np.asarray(X4, dtype=float), np.asarray(Y4, dtype=float)
    XI, ETA = np.meshgrid(xi, xi)                       # [b,a]: XI varies along a
    N00, N10 = (1 - XI) * (1 - ETA) / 4, (1 + XI) * (1 - ETA) / 4
    N01, N11 = (1 - XI) * (1 + ETA) / 4, (1 + XI) * (1 + ETA) / 4
    x = N00 * X4[0, 0] + N10 * X4[0, 1] + N01 * X4[1, 0] + N11 * X4[1, 1]
    y = N00 * Y4[0, 0] + N10 * Y4[0, 1] + N01 * Y4[1, 0] + N11 * Y4[1, 1]
    x_xi = ((1 - ETA) * (X4[0, 1] - X4[0, 0]) + (1 + ETA) * (X4[1, 1] - X4[1, 0])) / 4
    y_xi = ((1 - ETA) * (Y4[0, 1] - Y4[0, 0]) + (1 + ETA) * (Y4[1, 1] - Y4[1, 0])) / 4
    x_eta = ((1 - XI) * (X4[1, 0] - X4[0, 0]) + (1 + XI) * (X4[1, 1] - X4[0, 1])) / 4
    y_eta = ((1 - XI) * (Y4[1, 0] - Y4[0, 0]) + (1 + XI) * (Y4[1, 1] - Y4[0, 1])) / 4
    det = x_xi * y_eta - x_eta * y_xi
    if np.any(det <= 0):
        raise ValueError("element is not convex / not positively oriented")
    gxx = (x_eta ** 2 + y_eta ** 2) / det
    gxy = -(x_xi * x_eta + y_xi * y_eta) / det
    gyy = (x_xi ** 2 + y_xi ** 2) / det
    return x, y, det, gxx, gxy, gyy


def element_stiffness_quad(p: int, X4, Y4):
    """A_e[i,j] = sum_q w_q (grad phi_j . grad phi_i detJ)(q), local node (a,b) -> b*(p+1)+a, written
    as D^T (geometric factors) D."""
    _, w, D = gll(p)
    _, _, _, gxx, gxy, gyy = quad_geometry(p, X4, Y4)
    I = np.eye(p + 1)
    Dxi, Deta = np.kron(I, D), np.kron(D, I)            # d/dxi acts on a, d/deta on b
    W2 = np.outer(w, w)                                 # [b,a]
    Gxx, Gxy, Gyy = (np.diag((W2 * g).reshape(-1)) for g in (gxx, gxy, gyy))
    return Dxi.T @ Gxx @ Dxi + Dxi.T @ Gxy @ Deta + Deta.T @ Gxy @ Dxi + Deta.T @ Gyy @ Deta


def region_operators_quads(p: int, VX, VY):
    """Stiffness A (sparse), geometric lumped mass m[j,i] = sum_e w_a w_b detJ and geometric edge weights
    s[side] = sum_e w_a |edge_e|/2 of the region whose (ey+1) x (ex+1) vertices are VX, VY — the general-geometry
    counterpart of _region_operators."""
    VX, VY = np.asarray(VX, dtype=float), np.asarray(VY, dtype=float)
    ey, ex = VX.shape[0] - 1, VX.shape[1] - 1
    _, w, _ = gll(p)
    npx, npy = ex * p + 1, ey * p + 1
    rows, cols, vals = [], [], []
    m = np.zeros((npy, npx))
    la = np.arange(p + 1)
    for fy in range(ey):
        for fx in range(ex):
            X4, Y4 = VX[fy:fy + 2, fx:fx + 2], VY[fy:fy + 2, fx:fx + 2]
            Ae = element_stiffness_quad(p, X4, Y4)
            det = quad_geometry(p, X4, Y4)[2]
            gi = ((fy * p + la)[:, None] * npx + (fx * p + la)[None, :]).reshape(-1)
            rows.append(np.repeat(gi, (p + 1) ** 2))
            cols.append(np.tile(gi, (p + 1) ** 2))
            vals.append(Ae.reshape(-1))
            m[fy * p:fy * p + p + 1, fx * p:fx * p + p + 1] += np.outer(w, w) * det
    A = sp.csr_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))),
                      shape=(npx * npy, npx * npy))
    A.sum_duplicates()

    def side_weights(PX, PY):                           # polyline of vertices -> assembled w_a * |edge|/2
        out = np.zeros((len(PX) - 1) * p + 1)
        for e in range(len(PX) - 1):
            half = 0.5 * math.hypot(PX[e + 1] - PX[e], PY[e + 1] - PY[e])
            out[e * p:e * p + p + 1] += half * w
        return out
    s = [side_weights(VX[:, 0], VY[:, 0]), side_weights(VX[:, -1], VY[:, -1]),
         side_weights(VX[0, :], VY[0, :]), side_weights(VX[-1, :], VY[-1, :])]
    return A, m, s


def node_coords_quads(p: int, VX, VY):
    """(npy, npx) coordinates of the global GLL nodes of the mapped mesh."""
    VX, VY = np.asarray(VX, dtype=float), np.asarray(VY, dtype=float)
    ey, ex = VX.shape[0] - 1, VX.shape[1] - 1
    X = np.zeros((ey * p + 1, ex * p + 1))
    Y = np.zeros_like(X)
    for fy in range(ey):
        for fx in range(ex):
            x, y = quad_geometry(p, VX[fy:fy + 2, fx:fx + 2], VY[fy:fy + 2, fx:fx + 2])[:2]
            X[fy * p:fy * p + p + 1, fx * p:fx * p + p + 1] = x
            Y[fy * p:fy * p + p + 1, fx * p:fx * p + p + 1] = y
    return X, Y


def choose_nt_quads(p, VX, VY, c_nodes, omega, cfl_frac):
    """N_t for general quads (reading R24, the element-wise form of R9).  lmax(M^-1 A) <= max_e lmax(M_e^-1 A_e)
    (A and M are sums of element matrices), and on one element, with Lhat = Lambda_p / 4 the largest
    eigenvalue of the reference pencil (K, W) on [-1,1]:
        u^T A_e u <= sum_q w_q [(gxx+|gxy|) u_xi^2 + (gyy+|gxy|) u_eta^2] <= Lhat (Gx + Gy) sum_q w_q u_q^2,
        u^T M_e u >= mu sum_q w_q u_q^2,   Gx = max_q (gxx+|gxy|), Gy = max_q (gyy+|gxy|), mu = min_q detJ/c^2,
    so lmax <= max_e Lhat (Gx+Gy)/mu.  On hx-by-hy rectangles this is c_max^2 Lambda_p (1/hx^2+1/hy^2): choose_nt."""
    VX, VY = np.asarray(VX, dtype=float), np.asarray(VY, dtype=float)
    ey, ex = VX.shape[0] - 1, VX.shape[1] - 1
    c = np.asarray(c_nodes, dtype=float)
    lhat = lambda_p(p) / 4.0
    lmax = 0.0
    for fy in range(ey):
        for fx in range(ex):
            _, _, det, gxx, gxy, gyy = quad_geometry(p, VX[fy:fy + 2, fx:fx + 2], VY[fy:fy + 2, fx:fx + 2])
            ce = c[fy * p:fy * p + p + 1, fx * p:fx * p + p + 1]
            Gx, Gy = np.max(gxx + np.abs(gxy)), np.max(gyy + np.abs(gxy))
            mu = np.min(det / ce ** 2)
            lmax = max(lmax, lhat * (Gx + Gy) / mu)
    dt_stab = 2.0 / math.sqrt(lmax)
    T = 2.0 * math.pi / omega
    return max(4, int(math.ceil(T / (cfl_frac * dt_stab) * (1.0 - 1e-12))))
