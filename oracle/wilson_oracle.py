"""CPU oracle for the Wilson-loop hot path of BerryEasy (arXiv 2312.13051).

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this file.  It shares no code with the
CUDA path (``paper_2312_13051_b200/csrc``) and imports nothing from the product package.

Plain NumPy/LAPACK (float64 / complex128), explicit Python loops over k-points, written in the
order and notation of the paper.  Every function cites the passage it follows
(``PAPER.md:<line>`` = /root/reference/PAPER.md) and, where the paper is silent, ambiguous or
garbled, the reading taken (``R<n>`` = SURVEY.md section 8(c), restated in DESIGN.md "Readings").

Pins (tests/test_oracle_pins.py, ``-m "not gpu"``): SSH Berry phase 0/pi and the position-gauge
shift; Eq. 4 Chern number C = 1 also against the Berry-curvature integral Eq. 5;
Abelian loops against closed-form eigenvectors; brute-force index-loop products on 2x2 / 4x4;
BHZ spin-sector windings +-1 and block reduction when [H,S]=0; PSO eigenvalues +-1
(PAPER.md:156); BBH nested polarization 1/2 vs 0; gauge invariance; |lambda| -> 1; the supercell
folding identity; closed-form and folded spectra for the eigenvalues; zheev vs zheevd.
Parity unpinned: none of the functions below -- but the *outputs on disordered configs 3-5* have
no closed form and are pinned only through the clean-limit identities above.
"""
from __future__ import annotations

import numpy as np

TWO_PI = 2.0 * np.pi


# ---------------------------------------------------------------------------------------------
# S1: exact diagonalization at every k ("exact diagonalization of a discretized
# Hamiltonian at many points in reciprocal space"; R14: numpy.linalg.eigh = LAPACK zheevd)
# ---------------------------------------------------------------------------------------------
def eigh_batched(H: np.ndarray):
    """H [count][N][N] Hermitian -> (E [count][N] ascending, U [count][N][N] columns = vectors)."""
    H = np.asarray(H)
    count, N, _ = H.shape
    E = np.empty((count, N), dtype=np.float64)
    U = np.empty((count, N, N), dtype=np.complex128)
    for c in range(count):
        E[c], U[c] = np.linalg.eigh(H[c])
    return E, U


def occupied_frames(H_loop: np.ndarray, n_occ: int):
    """Step 1 of SURVEY 8(c): U_j = lowest n_occ eigenvectors at each of the N1 points (R8).

    Returns (frames list of [N][n_occ], mingap = min_j (E[n_occ] - E[n_occ-1]) or +inf)."""
    frames = []
    mingap = np.inf
    for j in range(H_loop.shape[0]):
        E, V = np.linalg.eigh(H_loop[j])
        frames.append(V[:, :n_occ])
        if n_occ < E.shape[0]:
            mingap = min(mingap, E[n_occ] - E[n_occ - 1])
    return frames, mingap


# ---------------------------------------------------------------------------------------------
# S2-S4: discretized, path-ordered Wilson loop (Eq. 2)
# ---------------------------------------------------------------------------------------------
def wilson_matrix(frames, close=None) -> np.ndarray:
    """W = prod_{j=0}^{N1-1} U_j^dagger U_{j+1}, with U_{N1} := Phi U_0.

    Eq. 2 read per R1 (exactly N1 factors, the last closing onto k+G, PAPER.md:40
    "periodic boundary conditions must be imposed along the path"), R2 (F is the m x m overlap
    matrix, path ordered), R3 (ordering of BASELINE.json north_star: W = prod_j
    U_j^dagger U_{j+1}; the paper's product is W^dagger, so xbar_n = -theta_n / 2 pi), R4 (no
    unitarization of links or of W) and R6 (``close`` = Phi, the [N] unit-modulus embedding
    phases e^{-i G.r}; None = periodic gauge, Phi = 1).
    """
    n1 = len(frames)
    m = frames[0].shape[1]
    last = frames[0] if close is None else np.asarray(close)[:, None] * frames[0]
    W = np.eye(m, dtype=np.complex128)
    for j in range(n1):
        nxt = frames[j + 1] if j + 1 < n1 else last
        W = W @ (frames[j].conj().T @ nxt)
    return W


def eigenphases(W: np.ndarray):
    """theta_n = arg lambda_n(W) sorted ascending in (-pi, pi], and |lambda_n| in the same order.

    PAPER.md:38 (Eq. 2: e^{i 2 pi xbar} are the eigenvalues), PAPER.md:127 (Eq. 8, "Im Ln");
    R4: general complex eigenvalues (LAPACK zgeev), only the angle is kept; R7: branch (-pi, pi].
    """
    lam = np.linalg.eigvals(W)
    th = np.angle(lam)
    th = np.where(th <= -np.pi, np.pi, th)
    order = np.argsort(th, kind="stable")
    return th[order], np.abs(lam)[order]


def window_frames(H_loop: np.ndarray, band_lo: int, band_hi: int):
    """NEXT-3 (PAPER.md:79 ``bands`` "the list of band indices"): frames of the bands
    [band_lo, band_hi) in ascending-energy order, U_j = V_j[:, band_lo:band_hi].

    Returns (frames, mingap) with mingap = min over the loop of the gaps at BOTH edges of the window,
    E[band_lo] - E[band_lo-1] (if band_lo > 0) and E[band_hi] - E[band_hi-1] (if band_hi < N)."""
    frames = []
    mingap = np.inf
    for j in range(H_loop.shape[0]):
        E, V = np.linalg.eigh(H_loop[j])
        frames.append(V[:, band_lo:band_hi])
        if band_lo > 0:
            mingap = min(mingap, E[band_lo] - E[band_lo - 1])
        if band_hi < E.shape[0]:
            mingap = min(mingap, E[band_hi] - E[band_hi - 1])
    return frames, mingap


def wilson_surface_window(H_grid: np.ndarray, band_lo: int, band_hi: int, direction: int, close=None):
    """``wilson_surface`` for the band window [band_lo, band_hi) instead of the lowest n_occ bands."""
    grid_ndim = H_grid.ndim - 3
    L = _loops_view(H_grid, grid_ndim, direction)
    m = band_hi - band_lo
    th = np.empty((L.shape[0], m))
    ab = np.empty((L.shape[0], m))
    mg = np.empty(L.shape[0])
    for b in range(L.shape[0]):
        frames, mg[b] = window_frames(L[b], band_lo, band_hi)
        th[b], ab[b] = eigenphases(wilson_matrix(frames, close))
    return th, ab, mg


def wilson_loop(H_loop: np.ndarray, n_occ: int, close=None):
    """One loop: H_loop [N1][N][N] -> (theta [n_occ], |lambda| [n_occ], mingap)."""
    frames, mingap = occupied_frames(H_loop, n_occ)
    th, ab = eigenphases(wilson_matrix(frames, close))
    return th, ab, mingap


def _loops_view(H_grid: np.ndarray, grid_ndim: int, direction: int):
    """Move grid axis ``direction`` (0-based among the grid axes that follow the batch axis) last
    and flatten batch and the other grid axes into one loop index (row-major order kept)."""
    H = np.asarray(H_grid)
    N = H.shape[-1]
    ax = 1 + direction
    Hm = np.moveaxis(H, ax, grid_ndim)  # batch, other grid axes..., loop axis, N, N
    n1 = Hm.shape[grid_ndim]
    return Hm.reshape(-1, n1, N, N)


def wilson_surface(H_grid: np.ndarray, n_occ: int, direction: int, close=None):
    """Hybrid WCC surface (Eq. 3, PAPER.md:77-83 ``WSurf``): one Wilson loop along
    grid axis ``direction`` for every other grid point and every batch entry.

    H_grid [batch][dims...][N][N]; returns (theta [loops][n_occ], abs [loops][n_occ],
    mingap [loops]) with loops enumerated row-major over (batch, remaining axes)."""
    grid_ndim = H_grid.ndim - 3
    L = _loops_view(H_grid, grid_ndim, direction)
    th = np.empty((L.shape[0], n_occ))
    ab = np.empty((L.shape[0], n_occ))
    mg = np.empty(L.shape[0])
    for b in range(L.shape[0]):
        th[b], ab[b], mg[b] = wilson_loop(L[b], n_occ, close)
    return th, ab, mg


# ---------------------------------------------------------------------------------------------
# S6: spin-resolved Wilson loop (section IV, ``WSpinSurf``)
# ---------------------------------------------------------------------------------------------
def projected_spin(U: np.ndarray, S: np.ndarray):
    """Reduced PSO U^dagger S U (m x m Hermitian): the non-zero block of P s P.
    ``S`` is a dense [N][N] operator or a real diagonal [N] (PAPER.md:170 ``op``)."""
    S = np.asarray(S)
    SU = S[:, None] * U if S.ndim == 1 else S @ U
    return U.conj().T @ SU


def spin_resolved_loop(H_loop: np.ndarray, n_occ: int, S, m_lo: int | None = None, close=None, band_lo: int = 0):
    """Wilson loop of the negative (lower) and positive (upper) eigenstates of the
    PSO.  R10: the split is by count m_lo (default n_occ/2) on ascending PSO eigenvalues; the
    closing link uses Phi U_0 V_0^sigma.

    ``band_lo`` > 0 (NEXT-3): the bands [band_lo, n_occ) instead of the lowest n_occ, m = n_occ - band_lo.

    Returns (theta_lo [m_lo], theta_hi [m-m_lo], pso [N1][m], abs_lo, abs_hi, mingap).
    """
    m = n_occ - band_lo
    if m_lo is None or m_lo < 0:
        m_lo = m // 2
    frames, mingap = window_frames(H_loop, band_lo, n_occ) if band_lo else occupied_frames(H_loop, n_occ)
    lo, hi = [], []
    pso = np.empty((len(frames), m))
    for j, U in enumerate(frames):
        sig, V = np.linalg.eigh(projected_spin(U, S))
        pso[j] = sig
        lo.append(U @ V[:, :m_lo])
        hi.append(U @ V[:, m_lo:])
    th_lo, ab_lo = eigenphases(wilson_matrix(lo, close))
    th_hi, ab_hi = eigenphases(wilson_matrix(hi, close))
    return th_lo, th_hi, pso, ab_lo, ab_hi, mingap


def spin_resolved_surface(H_grid, n_occ, direction, S, m_lo=None, close=None, band_lo: int = 0):
    """``WSpinSurf``: spin_resolved_loop for every transverse point / batch entry."""
    m = n_occ - band_lo
    if m_lo is None or m_lo < 0:
        m_lo = m // 2
    grid_ndim = H_grid.ndim - 3
    L = _loops_view(H_grid, grid_ndim, direction)
    B, n1 = L.shape[0], L.shape[1]
    th_lo = np.empty((B, m_lo))
    th_hi = np.empty((B, m - m_lo))
    pso = np.empty((B, n1, m))
    for b in range(B):
        th_lo[b], th_hi[b], pso[b], _, _, _ = spin_resolved_loop(L[b], n_occ, S, m_lo, close, band_lo)
    return th_lo, th_hi, pso


# ---------------------------------------------------------------------------------------------
# S5: nested Wilson loop (section III Eq. 8, PAPER.md:144-146 ``WNWL``)
# ---------------------------------------------------------------------------------------------
def branch_angle(lam: np.ndarray, theta_cut: float) -> np.ndarray:
    """arg(lam) on the branch (theta_cut - 2 pi, theta_cut]."""
    th = np.angle(lam)
    th = np.where(th > theta_cut, th - TWO_PI, th)
    th = np.where(th <= theta_cut - TWO_PI, th + TWO_PI, th)
    return th


def nested_wilson(H_plane: np.ndarray, n_occ: int, base: int = 0, wb_lo: int = 0, wb_hi: int = 1,
                  theta_cut: float = np.pi, close1=None, close2=None):
    """H_plane [N2][N1][N][N] (dir2 slow, dir1 fast) -> (theta1 [N2][n_occ], theta_nested [|S|]).

    Eq. 8: the Wannier Hamiltonian is Im Ln of the path-ordered loop along k1,
    "constructed numerically ... by replacing the right hand side of eq. (8) with the discretized
    formulation of the integral in eq. (2)"; its bands are then looped along k2.
    R9: for every k2 the first loop starts at index ``base`` on dir1; lambda, R = eig(W); Wannier
    bands ordered by theta on the branch (theta_cut - 2 pi, theta_cut]; V_S = right eigenvectors
    wb_lo..wb_hi-1, orthonormalized (QR; only their span matters); w(k2) = U_base(k2) V_S;
    second loop over k2 with closing phase Phi_2.
    """
    n2, n1 = H_plane.shape[0], H_plane.shape[1]
    theta1 = np.empty((n2, n_occ))
    wframes = []
    for i2 in range(n2):
        frames, _ = occupied_frames(H_plane[i2], n_occ)
        rolled = frames[base:] + frames[:base]
        # when the loop starts at ``base`` the closing frame is Phi_1 U_base and every frame that
        # was wrapped past the zone boundary carries Phi_1 as well (u(k+G) = Phi u(k), R6)
        if close1 is not None and base > 0:
            ph = np.asarray(close1)[:, None]
            rolled = frames[base:] + [ph * f for f in frames[:base]]
        W = wilson_matrix(rolled, close1)
        lam, R = np.linalg.eig(W)
        th = branch_angle(lam, theta_cut)
        order = np.argsort(th, kind="stable")
        th_pi = np.angle(lam)
        th_pi = np.where(th_pi <= -np.pi, np.pi, th_pi)
        theta1[i2] = np.sort(th_pi)
        VS = R[:, order[wb_lo:wb_hi]]
        Q, _ = np.linalg.qr(VS)
        wframes.append(rolled[0] @ Q)
    theta_n, _ = eigenphases(wilson_matrix(wframes, close2))
    return theta1, theta_n


# ---------------------------------------------------------------------------------------------
# NEXT-2: Berry flux through the plaquettes of a periodic grid ("integrated Berry
# flux through one plaquette", the coupling-matrix method on a 20 x 20 grid)
# ---------------------------------------------------------------------------------------------
def plaquette_flux(H_plane: np.ndarray, n_occ: int, S=None, m_lo: int | None = None):
    """H_plane [ny][nx][N][N] (periodic in both directions) -> flux [ny][nx] in (-pi, pi]:

        flux[j][i] = arg det( U_ji^+ U_j,i+1 . U_j,i+1^+ U_j+1,i+1 . U_j+1,i+1^+ U_j+1,i . U_j+1,i^+ U_ji ),

    the discretized loop of Eq. 2 around one plaquette, kx step first (links as in
    ``wilson_matrix``: R2, R3, R4 -- no unitarization; det makes the result gauge invariant).
    With ``S`` the frames are first rotated into the lower / upper PSO sectors (R10) and
    (flux_lo, flux_hi) is returned ("spin-resolved generalization of the coupling matrix method").
    sum(flux) / 2 pi is an integer: the Chern number in the orientation of the paper's Eq. 6 flow (R3).
    """
    ny, nx = H_plane.shape[:2]

    def frames_at(j, i):
        E, V = np.linalg.eigh(H_plane[j, i])
        U = V[:, :n_occ]
        if S is None:
            return (U,)
        Sm = np.asarray(S)
        SU = Sm[:, None] * U if Sm.ndim == 1 else Sm @ U
        sig, Vs = np.linalg.eigh(U.conj().T @ SU)
        ml = n_occ // 2 if m_lo is None else m_lo
        return (U @ Vs[:, :ml], U @ Vs[:, ml:])

    F = [[frames_at(j, i) for i in range(nx)] for j in range(ny)]
    nsec = len(F[0][0])
    out = [np.empty((ny, nx)) for _ in range(nsec)]
    for s in range(nsec):
        for j in range(ny):
            for i in range(nx):
                a, b = F[j][i][s], F[j][(i + 1) % nx][s]
                c, d = F[(j + 1) % ny][(i + 1) % nx][s], F[(j + 1) % ny][i][s]
                W = (a.conj().T @ b) @ (b.conj().T @ c) @ (c.conj().T @ d) @ (d.conj().T @ a)
                ph = np.angle(np.linalg.slogdet(W)[0])
                out[s][j, i] = np.pi if ph <= -np.pi else ph
    return out[0] if S is None else (out[0], out[1])


# ---------------------------------------------------------------------------------------------
# S7: invariants (Eq. 6)
# ---------------------------------------------------------------------------------------------
def wrap_pi(x):
    """Wrap to (-pi, pi]."""
    y = np.mod(np.asarray(x, dtype=np.float64) + np.pi, TWO_PI) - np.pi
    return np.where(y <= -np.pi, np.pi, y)


def winding(theta: np.ndarray) -> float:
    """wind = (1/2 pi) sum_i wrap(Theta_{i+1} - Theta_i), Theta_i = sum_n theta_n at transverse
    point i of a closed cycle (indices cyclic).  theta [n_transverse][m]."""
    Th = np.sum(np.asarray(theta), axis=1)
    d = wrap_pi(np.roll(Th, -1) - Th)
    return float(np.sum(d) / TWO_PI)


def chern_number(theta: np.ndarray) -> int:
    """Eq. 6 in the paper's sign convention: C = -wind because the library's W is
    the Hermitian conjugate of the paper's product (R3), xbar_n = -theta_n / 2 pi."""
    return int(np.rint(-winding(theta)))


def nested_polarization(theta_nested: np.ndarray) -> float:
    """p = (-sum theta / 2 pi) mod 1, rounded to the nearest multiple of 1/2, reduced mod 1."""
    p = (-np.sum(theta_nested) / TWO_PI) % 1.0
    return float((np.rint(2.0 * p) / 2.0) % 1.0)


# ---------------------------------------------------------------------------------------------
# R7 comparator: sorted points on the circle
# ---------------------------------------------------------------------------------------------
def circ_sorted_distance(a: np.ndarray, b: np.ndarray) -> float:
    """min over all cyclic shifts s of max_n circdist(a_n, b_{n+s}) for two ascending phase sets
    of equal length (radians).  Phases sitting at the branch cut re-label by a cyclic shift."""
    a = np.sort(np.asarray(a, dtype=np.float64))
    b = np.sort(np.asarray(b, dtype=np.float64))
    m = a.shape[0]
    best = np.inf
    for s in range(m):
        d = np.abs(wrap_pi(a - np.roll(b, -s)))
        best = min(best, float(np.max(d)) if m else 0.0)
    return 0.0 if m == 0 else best
