"""CPU ORACLE, 3-D hexahedral variant (Section VII.B).

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as oracle/hz_oracle.py: only tests/, smoke() and the
cpu_baseline / --impl reference legs may import it; it shares nothing with the CUDA path).

The paper repeats the 2-D method on uniform hexahedra with (P+1)^3 nodes per element: the same discretisation
 with tensor-product GLL nodes in three directions, the same subdomain problems with the impedance
transmission condition on all SIX faces, and the same WaveHoltz subdomain solver (Algorithm 1,
PAPER.md:160-183) — oracle/hz_oracle.py's `waveholtz_iteration` and `wh_tables` are dimension-independent and are
used as they are.  Plain fp64 numpy/scipy; operators are Kronecker products of assembled 1-D matrices.

Readings: R1-R23 carry over with "side" -> "face"; R9 becomes
N_t = ceil(T / (cfl dt_stab)), dt_stab = 2 / sqrt(c_max^2 Lambda_p (1/hx^2 + 1/hy^2 + 1/hz^2));
R13: lambda lives per (subdomain, face, face node) INCLUDING the face's edge and corner nodes; a DOF on a subdomain
edge sums its two faces, a corner DOF its three.

Conventions
  node (I,J,K), flat index (K*npy + J)*npx + I (x fastest).
  faces 0=W (I=0), 1=E (I=max), 2=S (J=0), 3=N (J=max), 4=B (K=0), 5=T (K=max); a face array is indexed
  (K,J) flat K*npy+J on W/E, (K,I) flat K*npx+I on S/N, (J,I) flat J*npx+I on B/T.

Pins (tests/test_oracle3d_pins.py): constants in the kernel of A, symmetry, volume / face areas, exact energy of a
polynomial field, 2-D limit (a z-independent field sees the 2-D operators), the N_t bound against the dense spectrum,
plane wave recovered at high order, WaveHoltz fixed point == direct solve, converged DDM == direct solve.
Nothing here is "parity unpinned".
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as spla

from oracle.hz_oracle import gll, lambda_p, stiffness_1d, waveholtz_iteration, wh_tables

FW, FE, FS, FN, FB, FT = range(6)
OPPOSITE = (FE, FW, FN, FS, FT, FB)


def assembled_1d(p: int, ne: int, h: float):
    """Assembled 1-D stiffness (2/h) K and lumped mass (h/2) w of ne elements of length h."""
    _, w, _ = gll(p)
    K = stiffness_1d(p)
    n = ne * p + 1
    Ka = np.zeros((n, n))
    wa = np.zeros(n)
    for e in range(ne):
        sl = slice(e * p, e * p + p + 1)
        Ka[sl, sl] += (2.0 / h) * K
        wa[sl] += (h / 2.0) * w
    return sp.csr_matrix(Ka), wa


@dataclass
class Problem3D:
    nx: int
    ny: int
    nz: int
    p: int
    box: tuple                    # (x0, y0, z0, x1, y1, z1)
    c_nodes: np.ndarray           # (npz, npy, npx) wave speed at the nodes
    omega: float
    f: np.ndarray                 # (npz, npy, npx) complex source at the nodes
    bc_lambda: list | None = None  # 6 complex face arrays (2-D, in the face order above) or None

    @property
    def h(self):
        x0, y0, z0, x1, y1, z1 = self.box
        return (x1 - x0) / self.nx, (y1 - y0) / self.ny, (z1 - z0) / self.nz

    @property
    def shape(self):
        return self.nz * self.p + 1, self.ny * self.p + 1, self.nx * self.p + 1

    def node_coords(self):
        xi, _, _ = gll(self.p)
        out = []
        for n, a, h in zip((self.nx, self.ny, self.nz), self.box[:3], self.h):
            out.append(np.concatenate([a + h * (e + (xi[:-1] + 1) / 2) for e in range(n)] + [[a + h * n]]))
        return out


def region_operators(p, ex, ey, ez, hx, hy, hz):
    """Stiffness A = Kx (x) Wy (x) Wz + Wx (x) Ky (x) Wz + Wx (x) Wy (x) Kz (sparse), lumped mass m[k,j,i] =
    wx_i wy_j wz_k and the face weights s[face] (2-D arrays: products of the two in-face 1-D masses) of a box of
    ex*ey*ez elements (PAPER.md:109-113 in three dimensions)."""
    Kx, wx = assembled_1d(p, ex, hx)
    Ky, wy = assembled_1d(p, ey, hy)
    Kz, wz = assembled_1d(p, ez, hz)
    Wx, Wy, Wz = sp.diags(wx), sp.diags(wy), sp.diags(wz)
    A = (sp.kron(Wz, sp.kron(Wy, Kx)) + sp.kron(Wz, sp.kron(Ky, Wx)) + sp.kron(Kz, sp.kron(Wy, Wx))).tocsr()
    m = wz[:, None, None] * wy[None, :, None] * wx[None, None, :]
    s = [np.outer(wz, wy), np.outer(wz, wy), np.outer(wz, wx), np.outer(wz, wx), np.outer(wy, wx), np.outer(wy, wx)]
    return A, m, s


def face_index(npx, npy, npz, face):
    """Flat region indices of the nodes of one face, as a 2-D array in the face-array order."""
    I, J, K = np.arange(npx), np.arange(npy), np.arange(npz)
    if face in (FW, FE):
        i = 0 if face == FW else npx - 1
        return (K[:, None] * npy + J[None, :]) * npx + i
    if face in (FS, FN):
        j = 0 if face == FS else npy - 1
        return (K[:, None] * npy + j) * npx + I[None, :]
    k = 0 if face == FB else npz - 1
    return (k * npy + J[:, None]) * npx + I[None, :]


def assemble_global(pr: Problem3D):
    """(A - i w H - w^2 M) u = b on the whole box (eq. (4))."""
    hx, hy, hz = pr.h
    A, m, s = region_operators(pr.p, pr.nx, pr.ny, pr.nz, hx, hy, hz)
    npz, npy, npx = pr.shape
    c = np.asarray(pr.c_nodes, dtype=float).reshape(-1)
    M = m.reshape(-1) / c ** 2
    H = np.zeros_like(M)
    b = np.asarray(pr.f, dtype=complex).reshape(-1) * m.reshape(-1)
    for face in range(6):
        idx = face_index(npx, npy, npz, face).reshape(-1)
        H[idx] += s[face].reshape(-1) / c[idx]
        if pr.bc_lambda is not None:
            b[idx] += s[face].reshape(-1) * np.asarray(pr.bc_lambda[face], dtype=complex).reshape(-1)
    return A, M, H, b


def direct_solve(pr: Problem3D):
    A, M, H, b = assemble_global(pr)
    K = (A.astype(complex) - sp.diags(1j * pr.omega * H + pr.omega ** 2 * M)).tocsc()
    return spla.splu(K).solve(b).reshape(pr.shape)


def residual(pr: Problem3D, u):
    A, M, H, b = assemble_global(pr)
    u = np.asarray(u, dtype=complex).reshape(-1)
    r = b - (A @ u - (1j * pr.omega * H + pr.omega ** 2 * M) * u)
    return float(np.linalg.norm(r) / np.linalg.norm(b))


def choose_nt(p, hx, hy, hz, c_max, omega, cfl_frac):
    """Reading R9 in three dimensions."""
    lmax = c_max ** 2 * lambda_p(p) * (1.0 / hx ** 2 + 1.0 / hy ** 2 + 1.0 / hz ** 2)
    dt_stab = 2.0 / math.sqrt(lmax)
    T = 2.0 * math.pi / omega
    return max(4, int(math.ceil(T / (cfl_frac * dt_stab) * (1.0 - 1e-12))))


@dataclass
class Subdomain3D:
    pos: tuple                   # (ix, iy, iz)
    off: tuple                   # global node offset (I0, J0, K0)
    shape: tuple                 # (npz, npy, npx)
    A: sp.csr_matrix
    M: np.ndarray
    H: np.ndarray
    bf: np.ndarray
    s: list
    k_face: list
    neighbour: list
    face_idx: list = field(default_factory=list)


@dataclass
class DDMState3D:
    pr: Problem3D
    grid: tuple                  # (sx, sy, sz)
    tab: object
    subs: list
    lam: list                    # lam[l][face]: complex 2-D face array
    u: list


def ddm_setup(pr: Problem3D, sx, sy, sz, cfl_frac=0.5, n_t=None) -> DDMState3D:
    """sx*sy*sz box subdomains of (nx/sx)*(ny/sy)*(nz/sz) elements; A_l, M_l from the subdomain's own elements,
    H_l on ALL six faces (interfaces carry the impedance operator)."""
    if pr.nx % sx or pr.ny % sy or pr.nz % sz:
        raise ValueError("subdomain grid must divide the element grid (reading R23)")
    ex, ey, ez = pr.nx // sx, pr.ny // sy, pr.nz // sz
    hx, hy, hz = pr.h
    A, m, s = region_operators(pr.p, ex, ey, ez, hx, hy, hz)
    npx, npy, npz = ex * pr.p + 1, ey * pr.p + 1, ez * pr.p + 1
    c = np.asarray(pr.c_nodes, dtype=float)
    f = np.asarray(pr.f, dtype=complex)
    if n_t is None:
        n_t = choose_nt(pr.p, hx, hy, hz, float(c.max()), pr.omega, cfl_frac)
    tab = wh_tables(n_t, pr.omega)
    subs = []
    for iz in range(sz):
        for iy in range(sy):
            for ix in range(sx):
                I0, J0, K0 = ix * ex * pr.p, iy * ey * pr.p, iz * ez * pr.p
                cl = c[K0:K0 + npz, J0:J0 + npy, I0:I0 + npx].reshape(-1)
                fl = f[K0:K0 + npz, J0:J0 + npy, I0:I0 + npx].reshape(-1)
                M = m.reshape(-1) / cl ** 2
                H = np.zeros_like(M)
                bf = fl * m.reshape(-1)
                lin = lambda a, b_, c_: (c_ * sy + b_) * sx + a   # noqa: E731
                nb = [lin(ix - 1, iy, iz) if ix > 0 else -1, lin(ix + 1, iy, iz) if ix < sx - 1 else -1,
                      lin(ix, iy - 1, iz) if iy > 0 else -1, lin(ix, iy + 1, iz) if iy < sy - 1 else -1,
                      lin(ix, iy, iz - 1) if iz > 0 else -1, lin(ix, iy, iz + 1) if iz < sz - 1 else -1]
                fidx, kface = [], []
                for face in range(6):
                    idx = face_index(npx, npy, npz, face)
                    fidx.append(idx)
                    H[idx.reshape(-1)] += s[face].reshape(-1) / cl[idx.reshape(-1)]
                    kface.append(pr.omega / cl[idx])
                    if nb[face] < 0 and pr.bc_lambda is not None:
                        full = np.asarray(pr.bc_lambda[face], dtype=complex)
                        if face in (FW, FE):
                            part = full[K0:K0 + npz, J0:J0 + npy]
                        elif face in (FS, FN):
                            part = full[K0:K0 + npz, I0:I0 + npx]
                        else:
                            part = full[J0:J0 + npy, I0:I0 + npx]
                        bf[idx.reshape(-1)] += (s[face] * part).reshape(-1)
                subs.append(Subdomain3D((ix, iy, iz), (I0, J0, K0), (npz, npy, npx), A, M, H, bf, s, kface, nb, fidx))
    lam = [[np.zeros(sd.face_idx[face].shape, dtype=complex) for face in range(6)] for sd in subs]
    u = [np.zeros(npx * npy * npz, dtype=complex) for _ in subs]
    return DDMState3D(pr, (sx, sy, sz), tab, subs, lam, u)


def ddm_cycle(st: DDMState3D, l: int, n_wh: int, warm_start: bool):
    """Algorithm 1 on subdomain l; g = -lambda - 2 i k u on interface faces (R3)."""
    sd = st.subs[l]
    b = sd.bf.copy()
    for face in range(6):
        if sd.neighbour[face] >= 0:
            b[sd.face_idx[face].reshape(-1)] += (sd.s[face] * st.lam[l][face]).reshape(-1)
    u = st.u[l].copy() if warm_start else np.zeros_like(st.u[l])
    for _ in range(n_wh):
        u = waveholtz_iteration(sd.A, sd.M, sd.H, b, u, st.pr.omega, st.tab)
    g = [None] * 6
    for face in range(6):
        if sd.neighbour[face] >= 0:
            g[face] = -st.lam[l][face] - 2j * sd.k_face[face] * u[sd.face_idx[face]]
    return u, g


def ddm_sweep(st: DDMState3D, n_wh: int, warm_start: bool, relax: float):
    L = len(st.subs)
    new_u, gs = [None] * L, [None] * L
    for l in range(L):
        new_u[l], gs[l] = ddm_cycle(st, l, n_wh, warm_start)
    new_lam = [[a.copy() for a in st.lam[l]] for l in range(L)]
    for l in range(L):
        for face in range(6):
            r = st.subs[l].neighbour[face]
            if r >= 0:
                o = OPPOSITE[face]
                new_lam[r][o] = (1.0 - relax) * st.lam[r][o] + relax * gs[l][face]
    st.lam, st.u = new_lam, new_u
    return st


def ddm_gather(st: DDMState3D):
    """Mean of the copies at nodes shared by several subdomains (R19)."""
    acc = np.zeros(st.pr.shape, dtype=complex)
    cnt = np.zeros(st.pr.shape)
    for l, sd in enumerate(st.subs):
        I0, J0, K0 = sd.off
        npz, npy, npx = sd.shape
        acc[K0:K0 + npz, J0:J0 + npy, I0:I0 + npx] += st.u[l].reshape(sd.shape)
        cnt[K0:K0 + npz, J0:J0 + npy, I0:I0 + npx] += 1.0
    return acc / cnt


def ddm_solve(pr: Problem3D, sx, sy, sz, n_outer, n_wh, warm_start=True, relax=0.5, cfl_frac=0.5, state=None):
    st = state if state is not None else ddm_setup(pr, sx, sy, sz, cfl_frac)
    for _ in range(n_outer):
        ddm_sweep(st, n_wh, warm_start, relax)
    return st
