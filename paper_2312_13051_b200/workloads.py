"""Seeded synthetic input generators for the five BASELINE.json workloads.

This module only *builds Hamiltonian grids* H(k) -- the input of the hot path.  It holds none of
the method's arithmetic (no eigensolve, no overlaps, no Wilson products, no phases) and is the one
module shared by the CUDA path's tests/bench and by ``oracle/`` (recipe
restated in DESIGN.md "Input recipe").

The paper's own workloads are PyBinding models and a DFT-derived
Wannier model, none of which is available; the models below take their shapes
(4-band toy models on 100x100 grids, O(20x20) supercells with disorder / impurities, a many-band
Wannier-like model) and stand in for them.

Conventions
-----------
* complex128 everywhere, periodic gauge (H(k+G) = H(k), closing phase Phi = 1) unless stated.
* ``np.kron(A, B)``: first factor is the slow index.
* RNG: ``numpy.random.default_rng([BASE_SEED, config_id, realization])``.
* Grid layout: ``[batch][dims...][N][N]``, last grid axis fastest, row-major H[r][c].

Every ``*_parts`` function returns a small set of dense host matrices from which H at any grid
point is a fixed linear combination with phase factors; ``assemble_*`` evaluates that combination
with either numpy (host, oracle side) or torch (device, to avoid shipping tens of GB over PCIe).
"""
from __future__ import annotations

import numpy as np

BASE_SEED = 20231213

s0 = np.eye(2, dtype=np.complex128)
sx = np.array([[0, 1], [1, 0]], dtype=np.complex128)
sy = np.array([[0, -1j], [1j, 0]], dtype=np.complex128)
sz = np.array([[1, 0], [0, -1]], dtype=np.complex128)
PAULI = (s0, sx, sy, sz)


def _rng(config_id: int, realization: int = 0, seed: int = BASE_SEED):
    return np.random.default_rng([seed, config_id, realization])


# --------------------------------------------------------------------------------------------
# two-band models used by the oracle pins
# --------------------------------------------------------------------------------------------
def qwz_eq4(kx: float, ky: float, M: float = 1.5) -> np.ndarray:
    """Chern insulator of PAPER.md:64 (Eq. 4): sin kx s1 + sin ky s2 + (cos kx + cos ky + M) s3."""
    return np.sin(kx) * sx + np.sin(ky) * sy + (np.cos(kx) + np.cos(ky) + M) * sz


def qwz_grid(n1: int, n2: int, M: float = 1.5) -> np.ndarray:
    """[n2 ky][n1 kx][2][2], kx_i = 2 pi i / n1, ky_j = 2 pi j / n2."""
    H = np.empty((n2, n1, 2, 2), dtype=np.complex128)
    for j in range(n2):
        for i in range(n1):
            H[j, i] = qwz_eq4(2 * np.pi * i / n1, 2 * np.pi * j / n2, M)
    return H


def ssh_loop(v: float, w: float, n1: int, position_gauge: bool = False):
    """SSH chain.  Periodic gauge: h(k) = [[0, v + w e^{-ik}], [c.c., 0]].

    Position gauge (sublattice B at r = 1/2): the same Hamiltonian conjugated by
    D(k) = diag(1, e^{-ik/2}), for which H(k + 2 pi) = Phi H(k) Phi^dagger with
    Phi = diag(1, e^{-i pi}) = e^{-i G r}.  Returns (H [n1][2][2], Phi [2] or None).
    """
    H = np.zeros((n1, 2, 2), dtype=np.complex128)
    for i in range(n1):
        k = 2 * np.pi * i / n1
        h = v + w * np.exp(-1j * k)
        if position_gauge:
            # D^dagger H D with D = diag(e^{i k r_alpha}), r = (0, 1/2): H[0,1] -> h e^{ik/2}
            h = h * np.exp(0.5j * k)  # = v e^{ik/2} + w e^{-ik/2}
        H[i, 0, 1] = h
        H[i, 1, 0] = np.conj(h)
    if position_gauge:
        r = np.array([0.0, 0.5])
        phi = np.exp(-1j * 2 * np.pi * r)
        return H, phi
    return H, None


# --------------------------------------------------------------------------------------------
# config 1: BHZ 4-band (BASELINE.json configs[0])
# --------------------------------------------------------------------------------------------
def bhz4(kx: float, ky: float, m: float = 1.0) -> np.ndarray:
    """sin kx kron(sx,sz) + sin ky kron(sy,s0) + (m - cos kx - cos ky) kron(sz,s0)."""
    return (np.sin(kx) * np.kron(sx, sz) + np.sin(ky) * np.kron(sy, s0)
            + (m - np.cos(kx) - np.cos(ky)) * np.kron(sz, s0))


def bhz4_spin_z() -> np.ndarray:
    """S_z = kron(s0, sz) = diag(1,-1,1,-1); real diagonal [4]."""
    return np.real(np.diag(np.kron(s0, sz))).copy()


def config1_grid(n1: int = 100, n2: int = 101, m: float = 1.0) -> np.ndarray:
    """[n2 ky][n1 kx][4][4]; loop direction = last grid axis (kx)."""
    H = np.empty((n2, n1, 4, 4), dtype=np.complex128)
    for j in range(n2):
        for i in range(n1):
            H[j, i] = bhz4(2 * np.pi * i / n1, 2 * np.pi * j / n2, m)
    return H


# --------------------------------------------------------------------------------------------
# config 2: BBH quadrupole (BASELINE.json configs[1])
# --------------------------------------------------------------------------------------------
def bbh_gammas():
    """Gamma_k = -kron(tau2, sigma_k) (k=1,2,3), Gamma_4 = kron(tau1, sigma0)."""
    g1 = -np.kron(sy, sx)
    g2 = -np.kron(sy, sy)
    g3 = -np.kron(sy, sz)
    g4 = np.kron(sx, s0)
    return g1, g2, g3, g4


def bbh(kx: float, ky: float, gamma: float = 0.5, lam: float = 1.0) -> np.ndarray:
    g1, g2, g3, g4 = bbh_gammas()
    return ((gamma + lam * np.cos(kx)) * g4 + lam * np.sin(kx) * g3
            + (gamma + lam * np.cos(ky)) * g2 + lam * np.sin(ky) * g1)


def config2_grid(n1: int = 100, n2: int = 100, gamma: float = 0.5, lam: float = 1.0) -> np.ndarray:
    """[n2 ky][n1 kx][4][4]."""
    H = np.empty((n2, n1, 4, 4), dtype=np.complex128)
    for j in range(n2):
        for i in range(n1):
            H[j, i] = bbh(2 * np.pi * i / n1, 2 * np.pi * j / n2, gamma, lam)
    return H


def position_gauge_plane(H: np.ndarray, r1, r2, shift1: int = 0) -> np.ndarray:
    """H [n2][n1][N][N] (periodic gauge) -> D^dagger H D with D(k) = diag(exp(i (k1 r1 + k2 r2))), the same
    model with orbital alpha at the position (r1, r2)[alpha] inside the unit cell:
    H(k + G_a) = Phi_a H(k) Phi_a^dagger with the closing phases Phi_a = exp(-2 pi i r_a).
    ``shift1``: the periodic-gauge grid is first rolled by ``shift1`` points along k1 (grid index i then
    stands for k1 = 2 pi (i + shift1) / n1 while D still uses 2 pi i / n1) -- the input of the base-point pin.
    Returns (H_pos, Phi_1, Phi_2)."""
    n2, n1 = H.shape[:2]
    r1 = np.asarray(r1, dtype=np.float64)
    r2 = np.asarray(r2, dtype=np.float64)
    Hs = np.roll(H, -shift1, axis=1) if shift1 else H
    out = np.empty_like(Hs)
    for j in range(n2):
        for i in range(n1):
            D = np.exp(2j * np.pi * (i / n1 * r1 + j / n2 * r2))
            out[j, i] = np.conj(D)[:, None] * Hs[j, i] * D[None, :]
    return out, np.exp(-2j * np.pi * r1), np.exp(-2j * np.pi * r2)


def bhz4_plus_band(kx: float, ky: float, m: float = 1.0) -> np.ndarray:
    """5 bands: the BHZ model of config 1 plus one occupied, trivial spin-down orbital
    eps(k) = -2.5 - 0.3 cos kx (decoupled).  With n_occ = 3 the PSO has the eigenvalues (-1, -1, +1): the
    spin sectors have the sizes 2 and 1 (an uneven split, m_lo = 2)."""
    H = np.zeros((5, 5), dtype=np.complex128)
    H[:4, :4] = bhz4(kx, ky, m)
    H[4, 4] = -2.5 - 0.3 * np.cos(kx)
    return H


def bhz4_plus_band_spin_z() -> np.ndarray:
    return np.array([1.0, -1.0, 1.0, -1.0, -1.0])


def bhz4_plus_band_grid(n1: int, n2: int) -> np.ndarray:
    H = np.empty((n2, n1, 5, 5), dtype=np.complex128)
    for j in range(n2):
        for i in range(n1):
            H[j, i] = bhz4_plus_band(2 * np.pi * i / n1, 2 * np.pi * j / n2)
    return H


def rotated_basis(H: np.ndarray, S_diag: np.ndarray, seed: int = 7):
    """The same model in a randomly rotated orbital basis: H' = R H R^dagger at every grid point and the DENSE
    spin operator S' = R diag(S) R^dagger (``op`` may be any Hermitian matrix)."""
    N = H.shape[-1]
    rng = _rng(90, seed)
    R, _ = np.linalg.qr(rng.normal(size=(N, N)) + 1j * rng.normal(size=(N, N)))
    Hr = R @ H @ R.conj().T
    Sr = (R * np.asarray(S_diag)[None, :]) @ R.conj().T
    return Hr, 0.5 * (Sr + Sr.conj().T)


# --------------------------------------------------------------------------------------------
# configs 3, 4: BHZ supercells with twisted boundary phases
# --------------------------------------------------------------------------------------------
def bhz_supercell_parts(L: int, onsite: np.ndarray | None = None, m: float = 1.0):
    """Dense pieces of the L x L BHZ supercell, N = 4 L^2, site (x, y) -> rows 4 (L x + y) .. +3.

    Returns (H_bulk, Bx, By): H(t1, t2) = H_bulk + e^{i 2 pi t1} Bx + e^{-i 2 pi t1} Bx^dagger
                                               + e^{i 2 pi t2} By + e^{-i 2 pi t2} By^dagger.
    H_bulk is Hermitian and contains every hop that stays inside the supercell plus the on-site
    blocks; Bx (By) holds the T_{+x} (T_{+y}) blocks of the hops that wrap around x (y).
    ``onsite``: optional [L][L][4][4] extra on-site blocks (disorder, impurities).
    """
    N = 4 * L * L
    Tx = np.kron(sx, sz) / 2j - np.kron(sz, s0) / 2
    Ty = np.kron(sy, s0) / 2j - np.kron(sz, s0) / 2
    M0 = m * np.kron(sz, s0)
    Hb = np.zeros((N, N), dtype=np.complex128)
    Bx = np.zeros((N, N), dtype=np.complex128)
    By = np.zeros((N, N), dtype=np.complex128)

    def blk(x, y):
        o = 4 * (L * x + y)
        return slice(o, o + 4)

    for x in range(L):
        for y in range(L):
            a = blk(x, y)
            Hb[a, a] += M0
            if onsite is not None:
                Hb[a, a] += onsite[x, y]
            # hop (x,y) -> (x+1,y): H[(x,y),(x+1,y)] = Tx
            b = blk((x + 1) % L, y)
            if x + 1 < L:
                Hb[a, b] += Tx
                Hb[b, a] += Tx.conj().T
            else:
                Bx[a, b] += Tx
            b = blk(x, (y + 1) % L)
            if y + 1 < L:
                Hb[a, b] += Ty
                Hb[b, a] += Ty.conj().T
            else:
                By[a, b] += Ty
    return Hb, Bx, By


def assemble_supercell(parts, t1, t2, xp=np):
    """H at twists (t1, t2) (scalars or broadcastable arrays shaped [..., 1, 1]) from the parts.

    ``xp`` is numpy or torch; with torch the parts must already be tensors on the target device.
    """
    Hb, Bx, By = parts
    two_pi = 2.0 * np.pi
    if xp is np:
        p1 = np.exp(1j * two_pi * np.asarray(t1))
        p2 = np.exp(1j * two_pi * np.asarray(t2))
        return (Hb + p1 * Bx + np.conj(p1) * Bx.conj().T + p2 * By + np.conj(p2) * By.conj().T)
    import torch
    p1 = torch.polar(torch.ones_like(t1), two_pi * t1)
    p2 = torch.polar(torch.ones_like(t2), two_pi * t2)
    return (Hb + p1 * Bx + p1.conj() * Bx.conj().transpose(-1, -2)
            + p2 * By + p2.conj() * By.conj().transpose(-1, -2))


def config3_onsite(L: int, realization: int, W: float = 2.0, seed: int = BASE_SEED) -> np.ndarray:
    """Anderson disorder: one scalar w ~ U[-W/2, W/2] per site times 1_4."""
    rng = _rng(3, realization, seed)
    w = rng.uniform(-W / 2, W / 2, size=(L, L))
    return w[:, :, None, None] * np.eye(4, dtype=np.complex128)


def config3_parts(realization: int, L: int = 10, W: float = 2.0, seed: int = BASE_SEED):
    return bhz_supercell_parts(L, config3_onsite(L, realization, W, seed))


def config4_onsite(L: int, frac: float = 0.05, h: float = 0.3, axis: str = "z",
                   realization: int = 0, seed: int = BASE_SEED) -> np.ndarray:
    """Random-sign Zeeman impurities h_s * h * kron(s0, s_axis) on a seeded ``frac`` of sites."""
    rng = _rng(4, realization, seed)
    nsite = L * L
    nimp = int(round(frac * nsite))
    sites = rng.choice(nsite, nimp, replace=False)
    signs = rng.choice([-1, 1], nimp)
    spin = {"x": sx, "y": sy, "z": sz}[axis]
    on = np.zeros((L, L, 4, 4), dtype=np.complex128)
    for s, sg in zip(sites, signs):
        on[s // L, s % L] = sg * h * np.kron(s0, spin)
    return on


def config4_parts(L: int = 20, axis: str = "z", realization: int = 0, seed: int = BASE_SEED):
    return bhz_supercell_parts(L, config4_onsite(L, axis=axis, realization=realization, seed=seed))


def supercell_spin_z(L: int) -> np.ndarray:
    """S_z = 1_{L^2} (x) kron(s0, sz): real diagonal [4 L^2]."""
    return np.tile(bhz4_spin_z(), L * L)


def supercell_grid(parts_list, n1: int, n2: int, t2_indices=None) -> np.ndarray:
    """Host grid [len(parts_list)][n2 or len(t2_indices)][n1][N][N]; t1_i = i/n1, t2_j = j/n2."""
    js = list(range(n2)) if t2_indices is None else list(t2_indices)
    N = parts_list[0][0].shape[0]
    H = np.empty((len(parts_list), len(js), n1, N, N), dtype=np.complex128)
    for r, parts in enumerate(parts_list):
        for a, j in enumerate(js):
            for i in range(n1):
                H[r, a, i] = assemble_supercell(parts, i / n1, j / n2)
    return H


def supercell_grid_torch(parts_list, n1: int, n2: int, device, t2_indices=None):
    """Same grid as ``supercell_grid`` assembled on ``device`` (torch), chunked per realization."""
    import torch
    js = list(range(n2)) if t2_indices is None else list(t2_indices)
    N = parts_list[0][0].shape[0]
    out = torch.empty((len(parts_list), len(js), n1, N, N), dtype=torch.complex128, device=device)
    t1 = (torch.arange(n1, dtype=torch.float64, device=device) / n1).view(n1, 1, 1)
    for r, parts in enumerate(parts_list):
        tp = tuple(torch.from_numpy(p).to(device) for p in parts)
        for a, j in enumerate(js):
            t2 = torch.full((1, 1, 1), j / n2, dtype=torch.float64, device=device)
            out[r, a] = assemble_supercell(tp, t1, t2, xp=torch)
    return out


# --------------------------------------------------------------------------------------------
# Eq. 9: chiral higher-order topological insulator, second validation model
# --------------------------------------------------------------------------------------------
def chiral_hoti(kx: float, ky: float, kz: float, delta0: float = 1.0) -> np.ndarray:
    """H(k)/t = sin kx s1 x t1 + sin ky s1 x t2 + sin kz s1 x t3 + (cos kx + cos ky + cos kz - 1.5) s3 x t0
    + Delta0 (cos kx - cos ky) s2 x t0, with A x B = np.kron(A, B) (R12: first factor slow)."""
    return (np.sin(kx) * np.kron(sx, sx) + np.sin(ky) * np.kron(sx, sy) + np.sin(kz) * np.kron(sx, sz)
            + (np.cos(kx) + np.cos(ky) + np.cos(kz) - 1.5) * np.kron(sz, s0)
            + delta0 * (np.cos(kx) - np.cos(ky)) * np.kron(sy, s0))


def chiral_hoti_spin() -> np.ndarray:
    """s = sigma_3 x tau_3 = diag(1, -1, -1, 1), as a real diagonal."""
    return np.real(np.diag(np.kron(sz, sz))).copy()


def chiral_hoti_grid(n1: int, n2: int, kzs, delta0: float = 1.0) -> np.ndarray:
    """[len(kzs)][n2 ky][n1 kx][4][4]; kz given in reduced units t3 (kz = 2 pi t3), loops run along kx."""
    H = np.empty((len(kzs), n2, n1, 4, 4), dtype=np.complex128)
    for a, t3 in enumerate(kzs):
        for j in range(n2):
            for i in range(n1):
                H[a, j, i] = chiral_hoti(2 * np.pi * i / n1, 2 * np.pi * j / n2, 2 * np.pi * t3, delta0)
    return H


# --------------------------------------------------------------------------------------------
# config 5: synthetic Wannier-like 64-orbital cubic model
# --------------------------------------------------------------------------------------------
def config5_half_space_vectors():
    """The 13 lattice vectors R in {-1,0,1}^3 \\ {0} whose first non-zero component is positive."""
    out = []
    for a in (-1, 0, 1):
        for b in (-1, 0, 1):
            for c in (-1, 0, 1):
                R = (a, b, c)
                if R == (0, 0, 0):
                    continue
                first = next(v for v in R if v != 0)
                if first > 0:
                    out.append(R)
    assert len(out) == 13
    return out


def config5_parts(norb_spatial: int = 32, delta: float = 3.0, soc: float = 0.3,
                  decay: float = 1.5, seed: int = BASE_SEED):
    """Returns (H0 [64][64] Hermitian, Rs [13][3] int, HR [13][64][64]).

    H(k) = H0 + sum_R (HR e^{i k.R} + h.c.).  Each block is
    e^{-|R|/decay} [kron(g0, s0) + soc * sum_a kron(g_a, s_a)], g = (N + iN)/sqrt(2 no) iid;
    the on-site block is the same form Hermitized plus kron(diag(-delta.., +delta..), s0).
    """
    rng = _rng(5, 0, seed)
    no = norb_spatial
    nrm = np.sqrt(2.0 * no)

    def block():
        B = np.zeros((2 * no, 2 * no), dtype=np.complex128)
        for a in range(4):
            g = (rng.standard_normal((no, no)) + 1j * rng.standard_normal((no, no))) / nrm
            B += (1.0 if a == 0 else soc) * np.kron(g, PAULI[a])
        return B

    B0 = block()
    H0 = 0.5 * (B0 + B0.conj().T)
    stag = np.concatenate([-delta * np.ones(no // 2), delta * np.ones(no - no // 2)])
    H0 = H0 + np.kron(np.diag(stag), s0)
    Rs = np.array(config5_half_space_vectors(), dtype=np.int64)
    HR = np.empty((len(Rs), 2 * no, 2 * no), dtype=np.complex128)
    for n, R in enumerate(Rs):
        HR[n] = np.exp(-np.linalg.norm(R) / decay) * block()
    return H0, Rs, HR


def assemble_config5(parts, k, xp=np):
    """H(k) for k = (kx, ky, kz) in radians (numpy scalars) from ``config5_parts``."""
    H0, Rs, HR = parts
    H = H0.copy()
    for n in range(len(Rs)):
        ph = np.exp(1j * float(np.dot(k, Rs[n])))
        H = H + ph * HR[n] + np.conj(ph) * HR[n].conj().T
    return H


def config5_grid(parts, nx: int, ny: int, nz: int, ix=None, iy=None) -> np.ndarray:
    """Host grid [len(ix)][len(iy)][nz][64][64]; k = 2 pi (i/nx, j/ny, l/nz); loops run along kz."""
    ix = list(range(nx)) if ix is None else list(ix)
    iy = list(range(ny)) if iy is None else list(iy)
    N = parts[0].shape[0]
    H = np.empty((len(ix), len(iy), nz, N, N), dtype=np.complex128)
    for a, i in enumerate(ix):
        for b, j in enumerate(iy):
            for l in range(nz):
                k = 2 * np.pi * np.array([i / nx, j / ny, l / nz])
                H[a, b, l] = assemble_config5(parts, k)
    return H


def config5_grid_torch(parts, nx: int, ny: int, nz: int, device, ix=None, iy=None):
    """Same grid as ``config5_grid`` assembled on ``device`` with torch (one kx slab at a time)."""
    import torch
    ix = list(range(nx)) if ix is None else list(ix)
    iy = list(range(ny)) if iy is None else list(iy)
    H0, Rs, HR = parts
    N = H0.shape[0]
    tH0 = torch.from_numpy(H0).to(device)
    tHR = torch.from_numpy(HR).to(device)
    tRs = torch.from_numpy(Rs).to(device=device, dtype=torch.float64)
    out = torch.empty((len(ix), len(iy), nz, N, N), dtype=torch.complex128, device=device)
    ky = 2 * np.pi * torch.tensor(iy, dtype=torch.float64, device=device) / ny
    kz = 2 * np.pi * torch.arange(nz, dtype=torch.float64, device=device) / nz
    for a, i in enumerate(ix):
        kx = 2 * np.pi * i / nx
        acc = tH0.expand(len(iy), nz, N, N).clone()
        for n in range(len(Rs)):
            ang = kx * tRs[n, 0] + ky[:, None] * tRs[n, 1] + kz[None, :] * tRs[n, 2]
            ph = torch.polar(torch.ones_like(ang), ang)[:, :, None, None]
            acc += ph * tHR[n] + ph.conj() * tHR[n].conj().T
        out[a] = acc
    return out
