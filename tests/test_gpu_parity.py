"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerances (BASELINE.json north_star, written here):
  eigenvalues      |dE| <= 1e-10 * ||H||_2
  WCC phases       <= 1e-8 in units of 2 pi, sorted points on the circle (R7 comparator), on loops
                   with a spectral gap
  invariants       equal as integers / half-integers
Eigenvectors, Wannier-band vectors, PSO eigenvectors and W itself are gauge dependent and are
checked only through residuals / orthonormality.
"""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import wilson_oracle as wo
from paper_2312_13051_b200 import workloads as wl

pytestmark = pytest.mark.gpu

E_TOL = 1e-10
PH_TOL = 1e-8  # units of 2 pi


@pytest.fixture(scope="module")
def ctx():
    from paper_2312_13051_b200.binding import Context
    c = Context()
    yield c
    c.close()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def phase_dist(a, b):
    """max over loops of the R7 circular distance, in units of 2 pi."""
    return max(wo.circ_sorted_distance(a[i], b[i]) for i in range(a.shape[0])) / (2 * np.pi)


def check_eigh(ctx, H, nv):
    E, U, info = ctx.eigh_batched(dev(H), nv, want_info=True)
    E, info = E.cpu().numpy(), info.cpu().numpy()
    U = U.cpu().numpy() if U is not None else None
    Eo, _ = wo.eigh_batched(H)
    assert info.max() == 0
    for c in range(H.shape[0]):
        nrm = max(np.abs(Eo[c]).max(), 1e-300)
        assert np.abs(E[c] - Eo[c]).max() <= E_TOL * nrm + 1e-300   # bisection resolves 0 to the smallest normal number
        assert np.all(np.diff(E[c]) >= 0)
        if nv:
            N = H.shape[1]
            assert np.linalg.norm(H[c] @ U[c] - U[c] * E[c][:nv]) <= 1e-11 * nrm * N
            assert np.linalg.norm(U[c].conj().T @ U[c] - np.eye(nv)) <= 1e-11 * N


# ------------------------------------------------------------------------------ S1
@pytest.mark.parametrize("N", [1, 2, 3, 4, 7, 8])
def test_eigh_jacobi_path(ctx, N):
    rng = np.random.default_rng(N)
    A = rng.standard_normal((37, N, N)) + 1j * rng.standard_normal((37, N, N))
    check_eigh(ctx, A + A.conj().transpose(0, 2, 1), N)


def test_eigh_jacobi_chiral_degenerate_models(ctx):
    """H3: E = +-eps doubly degenerate (BHZ, BBH) -- the case one-sided Jacobi on H itself misses."""
    check_eigh(ctx, wl.config1_grid(13, 9).reshape(-1, 4, 4), 4)
    check_eigh(ctx, wl.config2_grid(11, 6).reshape(-1, 4, 4), 2)


@pytest.mark.parametrize("N,nv", [(9, 9), (17, 17), (31, 10), (33, 33), (64, 32), (65, 65), (100, 37), (104, 104), (257, 128)])
def test_eigh_tridiagonal_path_random(ctx, N, nv):
    """sizes spanning several 32-panels / 64-blocks and ragged tails"""
    rng = np.random.default_rng(N)
    A = rng.standard_normal((3, N, N)) + 1j * rng.standard_normal((3, N, N))
    check_eigh(ctx, A + A.conj().transpose(0, 2, 1), nv)


def test_eigh_large_all_vectors(ctx):
    """N = 1000 with ALL eigenvectors, N = 641 (first size on the 32-wide panels) and N = 640 (last on the
    16-wide ones) with a ragged vector count: residual, orthonormality and eigenvalues at scale."""
    rng = np.random.default_rng(1000)
    for N, nv in ((1000, 1000), (641, 333), (640, 320)):
        A = rng.standard_normal((2, N, N)) + 1j * rng.standard_normal((2, N, N))
        check_eigh(ctx, A + A.conj().transpose(0, 2, 1), nv)


@pytest.mark.parametrize("N,nv", [(128, 128), (130, 65), (200, 77), (257, 257), (400, 200), (449, 1), (800, 800)])
def test_eigh_two_stage_path_random(ctx, N, nv):
    """be_set_eigh_algorithm(1): dense -> band (k_panel / k_ysum / k_fused) -> tridiagonal (k_chase), back-transform
    through both stages (k_q2 + compact WY); sizes with ragged last tiles, a ragged last panel and short last
    reflectors (N not a multiple of 64 / 8)."""
    rng = np.random.default_rng(N)
    A = rng.standard_normal((2, N, N)) + 1j * rng.standard_normal((2, N, N))
    H = A + A.conj().transpose(0, 2, 1)
    ctx.set_eigh_algorithm(1)
    try:
        check_eigh(ctx, H, nv)
    finally:
        ctx.set_eigh_algorithm(2)


def test_eigh_two_stage_structured_and_degenerate(ctx):
    """Two-stage path on what the one-stage tests cover: a sparse disordered supercell (rank-deficient panels:
    most of a panel's rows are exact zeros), the clean supercell (highly degenerate spectrum), the identity and a
    zero matrix (every reflector trivial), and both algorithms giving the same eigenvalues on the same input."""
    ctx.set_eigh_algorithm(1)
    try:
        H = wl.supercell_grid([wl.config3_parts(2, L=6)], 3, 2).reshape(-1, 144, 144)
        check_eigh(ctx, H, 72)
        Hc = wl.supercell_grid([wl.bhz_supercell_parts(6)], 2, 2).reshape(-1, 144, 144)
        check_eigh(ctx, Hc, 144)
        Z = np.zeros((2, 160, 160), complex)
        Z[1] = np.eye(160)
        E, U = ctx.eigh_batched(dev(Z), 160)
        assert np.abs(E.cpu().numpy()[0]).max() < 1e-300 and np.abs(E.cpu().numpy()[1] - 1).max() < 1e-14
        for c in range(2):
            Uc = U.cpu().numpy()[c]
            assert np.linalg.norm(Uc.conj().T @ Uc - np.eye(160)) < 1e-11 * 160
        rng = np.random.default_rng(5)
        A = rng.standard_normal((3, 320, 320)) + 1j * rng.standard_normal((3, 320, 320))
        Hd = dev(A + A.conj().transpose(0, 2, 1))
        E1, _ = ctx.eigh_batched(Hd, 0)
        ctx.set_eigh_algorithm(0)
        E0, _ = ctx.eigh_batched(Hd, 0)
        assert (E1 - E0).abs().max().item() < 1e-10 * E0.abs().max().item()
    finally:
        ctx.set_eigh_algorithm(2)
    with pytest.raises(RuntimeError):
        ctx.set_eigh_algorithm(3)


def test_eigh_degenerate_clean_supercell_and_identity(ctx):
    """H4: heavily degenerate spectra (clean supercell at t=0), plus diagonal / scaled identity."""
    pc = wl.bhz_supercell_parts(6)
    H = np.array([wl.assemble_supercell(pc, 0.0, 0.0), wl.assemble_supercell(pc, 0.5, 0.0),
                  wl.assemble_supercell(pc, 0.17, 0.4)])
    check_eigh(ctx, H, 72)
    D = np.zeros((2, 20, 20), dtype=complex)
    D[0] = 2.5 * np.eye(20)
    D[1] = np.diag(np.arange(20) % 3).astype(complex)
    check_eigh(ctx, D, 20)
    # the on-chip reduction forms its reflectors with in-line reciprocals: zero columns (tau = 0), an
    # all-zero matrix, and entries far from 1
    Z = np.zeros((4, 64, 64), dtype=complex)
    Z[1] = np.diag(np.linspace(-1, 1, 64))
    Z[1][5, 40] = Z[1][40, 5] = 0.25          # one coupled pair in an otherwise diagonal matrix
    rng = np.random.default_rng(64)
    A = rng.standard_normal((64, 64)) + 1j * rng.standard_normal((64, 64))
    Z[2] = 1e6 * (A + A.conj().T)
    Z[3] = 1e-6 * (A + A.conj().T)
    check_eigh(ctx, Z, 64)


def test_eigh_config3_and_config5_matrices(ctx):
    p3 = wl.config3_parts(1)
    H = np.array([wl.assemble_supercell(p3, i / 33, 5 / 32) for i in (0, 7, 20)])
    check_eigh(ctx, H, 200)
    p5 = wl.config5_parts()
    rng = np.random.default_rng(5)
    H = np.array([wl.assemble_config5(p5, 2 * np.pi * rng.uniform(0, 1, 3)) for _ in range(40)])
    check_eigh(ctx, H, 32)


def test_eigh_edge_cases(ctx):
    H = dev(wl.config1_grid(4, 3).reshape(-1, 4, 4))
    E, U = ctx.eigh_batched(H, 0)            # eigenvalues only
    assert U is None and E.shape == (12, 4)
    E0, U0 = ctx.eigh_batched(H[:0], 2)      # empty batch
    assert E0.shape == (0, 4)
    # only the upper triangle of the row-major input is read
    A = wl.assemble_config5(wl.config5_parts(), np.array([0.3, 0.2, 0.1]))[None]
    Au = A.copy()
    Au[0][np.tril_indices(64, -1)] = 123.0
    E1, _ = ctx.eigh_batched(dev(A), 0)
    E2, _ = ctx.eigh_batched(dev(Au), 0)
    assert torch.equal(E1, E2)


def test_numerical_trouble_comes_back_as_nan_not_as_numbers(ctx):
    """the Wilson entry points have no d_info.  A loop one of whose matrices cannot be diagonalized
    (here: a NaN entry; the same flag carries inverse-iteration / QR non-convergence) returns NaN phases, the
    other loops are untouched -- on the Jacobi + general path (N = 9 > 8 forces it), the blocked path and the
    spin-resolved call."""
    rng = np.random.default_rng(11)
    for N, m in ((9, 3), (144, 72)):
        if N == 9:
            H = _random_gapped_grid(12, 5, N=9, m=3, seed=4)
        else:
            H = wl.supercell_grid([wl.config3_parts(1, L=6)], 7, 5)[0]
        tho, _, _ = wo.wilson_surface(H[None], m, 1)
        Hb = H.copy()
        Hb[2, 3, 0, 1] = np.nan
        Hb[2, 3, 1, 0] = np.nan
        th, ab, mg = ctx.wilson_loop(dev(Hb[None]), m, 1)
        th = th.cpu().numpy()
        assert np.all(np.isnan(th[2]))
        good = [0, 1, 3, 4]
        assert np.all(np.isfinite(th[good])) and phase_dist(th[good], tho[good]) <= PH_TOL
    H = wl.supercell_grid([wl.config4_parts(6, axis="x")], 7, 4)[0]
    S = wl.supercell_spin_z(6)
    Hb = H.copy()
    Hb[1, 0, 5, 5] = np.inf
    lo, hi, pso = ctx.spin_resolved_wilson(dev(Hb[None]), 72, 1, dev(S))
    lo, hi = lo.cpu().numpy(), hi.cpu().numpy()
    assert np.all(np.isnan(lo[1])) and np.all(np.isnan(hi[1]))
    assert np.all(np.isfinite(lo[[0, 2, 3]])) and np.all(np.isfinite(hi[[0, 2, 3]]))


def test_error_codes(ctx):
    from paper_2312_13051_b200.binding import BerryEasyError
    H = dev(wl.config1_grid(4, 3)[None])
    with pytest.raises(BerryEasyError):
        ctx.wilson_loop(H, 5, 1)          # n_occ > N
    with pytest.raises(BerryEasyError):
        ctx.wilson_loop(H, 2, 2)          # dir out of range
    with pytest.raises(BerryEasyError):
        ctx.nested_wilson(H, 2, 1, 1)     # dir1 == dir2
    assert ctx.lib.be_eigh_batched(ctx._h, None, 1, 4, 4, None, None, None) == -1


# ------------------------------------------------------------------------------ config 1 (full size)
def test_config1_full_wilson_and_spin_resolved(ctx):
    H = wl.config1_grid()[None]                       # [1][101][100][4][4]
    th, ab, mg = ctx.wilson_loop(dev(H), 2, 1)
    tho, abo, mgo = wo.wilson_surface(H, 2, 1)
    th, ab, mg = th.cpu().numpy(), ab.cpu().numpy(), mg.cpu().numpy()
    assert mgo.min() > 1.9
    assert np.abs(mg - mgo).max() < 1e-12
    assert phase_dist(th, tho) <= PH_TOL
    assert np.abs(np.sort(ab, 1) - np.sort(abo, 1)).max() < 1e-10
    S = wl.bhz4_spin_z()
    lo, hi, pso = ctx.spin_resolved_wilson(dev(H), 2, 1, dev(S))
    loo, hio, psoo = wo.spin_resolved_surface(H, 2, 1, S)
    assert phase_dist(lo.cpu().numpy(), loo) <= PH_TOL
    assert phase_dist(hi.cpu().numpy(), hio) <= PH_TOL
    assert np.abs(pso.cpu().numpy() - psoo).max() < 1e-10
    # invariants, exact: total winding 0, sectors +-1 (device winding kernel vs oracle)
    w = ctx.winding(torch.stack([th_.reshape(101, -1) for th_ in (lo, hi)])).cpu().numpy()
    assert [int(round(x)) for x in w] == [int(round(wo.winding(loo))), int(round(wo.winding(hio)))] == [1, -1]
    wt = ctx.winding(torch.from_numpy(th).cuda().reshape(1, 101, 2)).cpu().numpy()
    assert int(round(wt[0])) == int(round(wo.winding(tho))) == 0
    assert np.abs(w - np.rint(w)).max() < 1e-9


def test_qwz_chern_number_device(ctx):
    H = wl.qwz_grid(100, 100)[None]
    th, _, _ = ctx.wilson_loop(dev(H), 1, 1)
    tho, _, _ = wo.wilson_surface(H, 1, 1)
    assert phase_dist(th.cpu().numpy(), tho) <= PH_TOL
    w = ctx.winding(th.reshape(1, 100, 1)).cpu().numpy()[0]
    assert int(round(-w)) == wo.chern_number(tho) == 1


def test_loop_direction_and_batch_axes(ctx):
    """dir = 0 (loops strided in memory), 3 grid axes, batch > 1."""
    p5 = wl.config5_parts(norb_spatial=8)
    H = wl.config5_grid(p5, 5, 4, 6, ix=range(5), iy=range(4))      # [5][4][6][16][16]
    H4 = np.stack([H, H[::-1].copy()])                              # batch 2, ndim 3
    for d in (0, 1, 2):
        th, _, _ = ctx.wilson_loop(dev(H4), 8, d)
        tho, _, _ = wo.wilson_surface(H4, 8, d)
        assert phase_dist(th.cpu().numpy(), tho) <= PH_TOL


def test_closing_phase_position_gauge(ctx):
    for v, w_ in ((1.0, 0.5), (0.5, 1.0)):
        H, phi = wl.ssh_loop(v, w_, 50, position_gauge=True)
        th, _, _ = ctx.wilson_loop(dev(H[None]), 1, 0, close=dev(phi))
        tho, _, _ = wo.wilson_loop(H, 1, close=phi)
        assert abs(wo.wrap_pi(th.cpu().numpy()[0, 0] - tho[0])) / (2 * np.pi) <= PH_TOL
    # multi-band: supercell in the position gauge along x with Phi = exp(-i 2 pi x / L)
    L, n1 = 3, 7
    parts = wl.bhz_supercell_parts(L)
    xs = np.repeat(np.arange(L), L * 4).astype(float)
    Hl = []
    for i in range(n1):
        D = np.exp(1j * 2 * np.pi * (i / n1) * xs / L)
        Hl.append((np.conj(D)[:, None] * wl.assemble_supercell(parts, i / n1, 0.37)) * D[None, :])
    Hl = np.array(Hl)
    phi = np.exp(-1j * 2 * np.pi * xs / L)
    th, _, _ = ctx.wilson_loop(dev(Hl[None]), 18, 0, close=dev(phi))
    tho, _, _ = wo.wilson_loop(Hl, 18, close=phi)
    assert phase_dist(th.cpu().numpy(), tho[None]) <= PH_TOL


def test_degenerate_loops_single_point_and_full_filling(ctx):
    H = wl.config1_grid(1, 3)[None]                   # N1 = 1: W = U^dagger U = 1
    th, ab, mg = ctx.wilson_loop(dev(H), 2, 1)
    assert np.abs(th.cpu().numpy()).max() < 1e-12 and np.abs(ab.cpu().numpy() - 1).max() < 1e-12
    H = wl.config1_grid(9, 2)[None]                   # n_occ = N: every link unitary, mingap = +inf
    th, ab, mg = ctx.wilson_loop(dev(H), 4, 1)
    tho, abo, _ = wo.wilson_surface(H, 4, 1)
    assert phase_dist(th.cpu().numpy(), tho) <= PH_TOL
    assert np.abs(ab.cpu().numpy() - 1).max() < 1e-12 and np.all(np.isinf(mg.cpu().numpy()))


# ------------------------------------------------------------------------------ config 2 (full size)
def test_config2_full_nested_polarization(ctx):
    H = wl.config2_grid()                              # [100][100][4][4]
    th1, thn = ctx.nested_wilson(dev(H[None]), 2, 1, 0)
    th1o, thno = wo.nested_wilson(H, 2)
    assert phase_dist(th1.cpu().numpy()[0], th1o) <= PH_TOL
    thn = thn.cpu().numpy()[0]
    assert wo.circ_sorted_distance(thn, thno) / (2 * np.pi) <= PH_TOL
    assert wo.nested_polarization(thn) == wo.nested_polarization(thno) == 0.5


@pytest.mark.parametrize("gamma,p", [(0.5, 0.5), (1.5, 0.0)])
def test_nested_variants(ctx, gamma, p):
    H = wl.config2_grid(30, 24, gamma=gamma)
    for base, band in ((0, 1), (7, 0)):
        th1, thn = ctx.nested_wilson(dev(H[None]), 2, 1, 0, base=base, wb_lo=band, wb_hi=band + 1)
        th1o, thno = wo.nested_wilson(H, 2, base=base, wb_lo=band, wb_hi=band + 1)
        assert phase_dist(th1.cpu().numpy()[0], th1o) <= PH_TOL
        assert wo.circ_sorted_distance(thn.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL
        assert wo.nested_polarization(thn.cpu().numpy()[0]) == p
    # both Wannier bands: nested phases of the full occupied space
    th1, thn = ctx.nested_wilson(dev(H[None]), 2, 1, 0, wb_lo=0, wb_hi=2)
    _, thno = wo.nested_wilson(H, 2, wb_lo=0, wb_hi=2)
    assert wo.circ_sorted_distance(thn.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL
    # dir1 = 0, dir2 = 1 on the transposed grid gives the same numbers
    Ht = np.ascontiguousarray(H.transpose(1, 0, 2, 3))
    _, thn_t = ctx.nested_wilson(dev(Ht[None]), 2, 0, 1)
    _, thno = wo.nested_wilson(H, 2)
    assert wo.circ_sorted_distance(thn_t.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL


def test_nested_closing_phases_base_and_cut_on_device(ctx):
    """d_close1 / d_close2 / base / theta_cut of be_nested_wilson:
    BBH in a position gauge (asymmetric orbital positions, generic gamma), loops started at base = 5 so that
    wrapped frames carry Phi_1; the chiral position gauge whose nested polarization is exactly 1/2 + 0.1; and
    the chiral HOTI slice whose two Wannier bands are re-numbered by the cut."""
    n = 14
    H = wl.config2_grid(n, n, gamma=0.7)
    r1 = np.array([0.11, 0.37, -0.23, 0.41])
    r2 = np.array([0.29, -0.13, 0.07, 0.33])
    Hp, c1, c2 = wl.position_gauge_plane(H, r1, r2)
    for base, band in ((0, 0), (5, 1), (13, 0)):
        th1, thn = ctx.nested_wilson(dev(Hp[None]), 2, 1, 0, base=base, wb_lo=band, wb_hi=band + 1,
                                     close1=dev(c1), close2=dev(c2))
        th1o, thno = wo.nested_wilson(Hp, 2, base=base, wb_lo=band, wb_hi=band + 1, close1=c1, close2=c2)
        assert phase_dist(th1.cpu().numpy()[0], th1o) <= PH_TOL
        assert wo.circ_sorted_distance(thn.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL
    # only one of the two phases
    th1, thn = ctx.nested_wilson(dev(Hp[None]), 2, 1, 0, base=3, close2=dev(c2))
    th1o, thno = wo.nested_wilson(Hp, 2, base=3, close2=c2)
    assert phase_dist(th1.cpu().numpy()[0], th1o) <= PH_TOL
    assert wo.circ_sorted_distance(thn.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL
    # exact value: chiral position gauge along k2, p = 1/2 + 0.1 (tests/test_oracle_pins.py)
    Hb = wl.config2_grid(24, 24, gamma=0.5)
    r = np.array([0.3, 0.3, -0.1, -0.1])
    Hy, _, cy = wl.position_gauge_plane(Hb, np.zeros(4), r)
    _, thn = ctx.nested_wilson(dev(Hy[None]), 2, 1, 0, close2=dev(cy))
    assert abs(((-thn.cpu().numpy()[0, 0] / (2 * np.pi)) % 1.0) - 0.6) < 1e-8
    # n_occ > 2 (general Wannier-band path) with closing phases and a base point
    Hc = _coupled_bbh_grid(12, 10)
    r1 = np.linspace(-0.3, 0.4, 8); r2 = np.linspace(0.25, -0.35, 8)
    Hcp, c1, c2 = wl.position_gauge_plane(Hc, r1, r2)
    th1o, thno = wo.nested_wilson(Hcp, 4, base=4, wb_lo=0, wb_hi=2, close1=c1, close2=c2)
    th1, thn = ctx.nested_wilson(dev(Hcp[None]), 4, 1, 0, base=4, wb_lo=0, wb_hi=2, close1=dev(c1), close2=dev(c2))
    assert phase_dist(th1.cpu().numpy()[0], th1o) <= PH_TOL
    assert wo.circ_sorted_distance(thn.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL
    # theta_cut: the cut at 0 swaps the numbers of the two Wannier bands of the chiral HOTI slice
    Hz = wl.chiral_hoti_grid(16, 16, [0.1], 1.0)
    for cut in (0.0, np.pi, -1.0):
        for band in (0, 1):
            _, thn = ctx.nested_wilson(dev(Hz), 2, 1, 0, wb_lo=band, wb_hi=band + 1, theta_cut=cut)
            _, thno = wo.nested_wilson(Hz[0], 2, wb_lo=band, wb_hi=band + 1, theta_cut=cut)
            assert wo.circ_sorted_distance(thn.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL
    _, a = ctx.nested_wilson(dev(Hz), 2, 1, 0, wb_lo=0, wb_hi=1, theta_cut=0.0)
    _, b = ctx.nested_wilson(dev(Hz), 2, 1, 0, wb_lo=1, wb_hi=2, theta_cut=np.pi)
    _, c = ctx.nested_wilson(dev(Hz), 2, 1, 0, wb_lo=0, wb_hi=1, theta_cut=np.pi)
    assert abs(wo.wrap_pi(a.cpu().numpy()[0, 0] - b.cpu().numpy()[0, 0])) < 1e-8
    assert abs(wo.wrap_pi(a.cpu().numpy()[0, 0] - c.cpu().numpy()[0, 0])) > 0.1


def test_spin_resolved_uneven_split_and_dense_spin_operator_on_device(ctx):
    """m_lo != m / 2 at a real PSO gap and a dense Hermitian S (R10): BHZ plus one occupied
    spin-down orbital, n_occ = 3, sectors of 2 and 1; the same model in a rotated basis (dense S); and a
    spin-mixing supercell with an uneven split at its PSO gap."""
    n1, n2 = 40, 21
    H = wl.bhz4_plus_band_grid(n1, n2)
    S = wl.bhz4_plus_band_spin_z()
    loo, hio, psoo = wo.spin_resolved_surface(H[None], 3, 1, S, m_lo=2)
    lo, hi, pso = ctx.spin_resolved_wilson(dev(H[None]), 3, 1, dev(S), m_lo=2)
    assert lo.shape == (n2, 2) and hi.shape == (n2, 1)
    assert np.abs(pso.cpu().numpy() - psoo).max() < 1e-10
    assert phase_dist(lo.cpu().numpy(), loo) <= PH_TOL and phase_dist(hi.cpu().numpy(), hio) <= PH_TOL
    w_lo, w_hi = ctx.winding(lo[None]).item(), ctx.winding(hi[None]).item()
    assert abs(abs(w_lo) - 1) < 1e-9 and abs(w_lo + w_hi) < 1e-9
    Hr, Sr = wl.rotated_basis(H, S)
    loo_r, hio_r, psoo_r = wo.spin_resolved_surface(Hr[None], 3, 1, Sr, m_lo=2)      # the oracle's dense-S branch
    lo_r, hi_r, pso_r = ctx.spin_resolved_wilson(dev(Hr[None]), 3, 1, dev(Sr), m_lo=2)
    assert np.abs(pso_r.cpu().numpy() - psoo_r).max() < 1e-10
    assert phase_dist(lo_r.cpu().numpy(), loo_r) <= PH_TOL and phase_dist(hi_r.cpu().numpy(), hio_r) <= PH_TOL
    assert phase_dist(lo_r.cpu().numpy(), loo) <= PH_TOL                               # = the diagonal-S result
    # blocked eigensolver + DMMA GEMM path: spin-mixing N = 144 supercell plus three decoupled occupied spin-down
    # levels (N = 147, n_occ = 75): the PSO has 39 negative and 36 positive eigenvalues, gapped around 0
    parts = wl.config4_parts(6, axis="x")
    H0 = wl.supercell_grid([parts], 9, 4, t2_indices=[1, 2])
    Hs = np.zeros(H0.shape[:3] + (147, 147), complex)
    Hs[..., :144, :144] = H0
    for q in range(3):
        Hs[..., 144 + q, 144 + q] = -4.0 - 0.1 * q
    Ss = np.concatenate([wl.supercell_spin_z(6), -np.ones(3)])
    _, _, p0 = wo.spin_resolved_surface(Hs, 75, 1, Ss)
    assert np.all((p0 < 0).sum(axis=-1) == 39) and np.abs(p0).min() > 0.05             # a gap at the count 39 everywhere
    loo, hio, psoo = wo.spin_resolved_surface(Hs, 75, 1, Ss, m_lo=39)
    lo, hi, pso = ctx.spin_resolved_wilson(dev(Hs), 75, 1, dev(Ss), m_lo=39)
    assert lo.shape == (2, 39) and hi.shape == (2, 36)
    assert np.abs(pso.cpu().numpy() - psoo).max() < 1e-10
    assert phase_dist(lo.cpu().numpy(), loo) <= PH_TOL and phase_dist(hi.cpu().numpy(), hio) <= PH_TOL


def _coupled_bbh_grid(n1, n2, eps=0.05, seed=3):
    """Two BBH copies (gamma = 0.5, 0.6) weakly coupled: N = 8, n_occ = 4, Wannier gap ~0.8."""
    rng = np.random.default_rng(seed)
    C = rng.standard_normal((4, 4)) + 1j * rng.standard_normal((4, 4))
    H = np.zeros((n2, n1, 8, 8), complex)
    for j in range(n2):
        for i in range(n1):
            kx, ky = 2 * np.pi * i / n1, 2 * np.pi * j / n2
            H[j, i, :4, :4] = wl.bbh(kx, ky, 0.5, 1.0)
            H[j, i, 4:, 4:] = wl.bbh(kx, ky, 0.6, 1.0)
            H[j, i, :4, 4:] = eps * C
            H[j, i, 4:, :4] = eps * C.conj().T
    return H


def _random_gapped_grid(n1, n2, N=7, m=3, seed=0):
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    A0 = np.diag([-2.0] * m + [2.0] * (N - m)) + 0.15 * (A + A.conj().T)
    T = [0.25 * (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))) for _ in range(2)]
    H = np.zeros((n2, n1, N, N), complex)
    for j in range(n2):
        for i in range(n1):
            kx, ky = 2 * np.pi * i / n1, 2 * np.pi * j / n2
            H[j, i] = (A0 + T[0] * np.exp(1j * kx) + T[0].conj().T * np.exp(-1j * kx)
                       + T[1] * np.exp(1j * ky) + T[1].conj().T * np.exp(-1j * ky))
    return H


def test_nested_general_n_occ_above_two(ctx):
    """S5 beyond the closed-form 2 x 2 case: Wannier-band vectors by inverse iteration on W - lambda I."""
    H = _coupled_bbh_grid(24, 20)
    th1o, thno = wo.nested_wilson(H, 4, wb_lo=0, wb_hi=2)
    assert (th1o[:, 2] - th1o[:, 1]).min() > 0.5                      # Wannier gap between the selected pair and the rest
    th1, thn = ctx.nested_wilson(dev(H[None]), 4, 1, 0, wb_lo=0, wb_hi=2)
    assert phase_dist(th1.cpu().numpy()[0], th1o) <= PH_TOL
    assert wo.circ_sorted_distance(thn.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL
    # upper pair, other base point
    th1o, thno = wo.nested_wilson(H, 4, base=5, wb_lo=2, wb_hi=4)
    th1, thn = ctx.nested_wilson(dev(H[None]), 4, 1, 0, base=5, wb_lo=2, wb_hi=4)
    assert phase_dist(th1.cpu().numpy()[0], th1o) <= PH_TOL
    assert wo.circ_sorted_distance(thn.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL
    # odd sizes, a single non-degenerate middle band
    H = _random_gapped_grid(20, 16)
    th1o, thno = wo.nested_wilson(H, 3, wb_lo=1, wb_hi=2)
    assert min((th1o[:, 1] - th1o[:, 0]).min(), (th1o[:, 2] - th1o[:, 1]).min()) > 0.05
    th1, thn = ctx.nested_wilson(dev(H[None]), 3, 1, 0, wb_lo=1, wb_hi=2)
    assert phase_dist(th1.cpu().numpy()[0], th1o) <= PH_TOL
    assert wo.circ_sorted_distance(thn.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL
    # all bands selected: the nested loop of the whole occupied space = plain loop along dir2 at fixed base
    th1, thn = ctx.nested_wilson(dev(H[None]), 3, 1, 0, wb_lo=0, wb_hi=3)
    _, thno = wo.nested_wilson(H, 3, wb_lo=0, wb_hi=3)
    assert wo.circ_sorted_distance(thn.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL
    # larger occupied space (disordered BHZ supercell, N = 64, n_occ = 32), all 32 Wannier bands: the
    # Hessenberg-QR + LU path at a size spanning several tiles; the span is the whole occupied space
    H = wl.supercell_grid([wl.config3_parts(1, L=4)], 9, 6)[0]
    th1o, thno = wo.nested_wilson(H, 32, wb_lo=0, wb_hi=32)
    th1, thn = ctx.nested_wilson(dev(H[None]), 32, 1, 0, wb_lo=0, wb_hi=32)
    assert phase_dist(th1.cpu().numpy()[0], th1o) <= PH_TOL
    assert wo.circ_sorted_distance(thn.cpu().numpy()[0], thno) / (2 * np.pi) <= PH_TOL


# ------------------------------------------------------------------------------ config 3 (reduced)
def test_config3_reduced_disordered_supercell(ctx):
    """N = 400, n_occ = 200, 2 realizations x 2 t2 x 33 t1 (full loop length, full matrix size)."""
    parts = [wl.config3_parts(r) for r in (0, 5)]
    H = wl.supercell_grid(parts, 33, 32, t2_indices=[0, 13])
    th, ab, mg = ctx.wilson_loop(dev(H), 200, 1)
    tho, abo, mgo = wo.wilson_surface(H, 200, 1)
    assert mgo.min() > 0.1
    assert np.abs(mg.cpu().numpy() - mgo).max() < 1e-10 * 4
    assert phase_dist(th.cpu().numpy(), tho) <= PH_TOL
    assert np.abs(np.sort(ab.cpu().numpy(), 1) - np.sort(abo, 1)).max() < 1e-9


# ------------------------------------------------------------------------------ config 4 (reduced)
def test_config4_reduced_spin_resolved_supercell(ctx):
    """L = 8 (N = 256, sectors of 64) full loop length, z impurities ([H,S]=0) and x impurities."""
    for axis in ("z", "x"):
        parts = wl.config4_parts(8, axis=axis)
        H = wl.supercell_grid([parts], 25, 24, t2_indices=[0, 11])
        S = wl.supercell_spin_z(8)
        lo, hi, pso = ctx.spin_resolved_wilson(dev(H), 128, 1, dev(S))
        loo, hio, psoo = wo.spin_resolved_surface(H, 128, 1, S)
        assert np.abs(pso.cpu().numpy() - psoo).max() < 1e-10
        assert phase_dist(lo.cpu().numpy(), loo) <= PH_TOL
        assert phase_dist(hi.cpu().numpy(), hio) <= PH_TOL
        if axis == "z":
            assert np.abs(np.abs(psoo) - 1).max() < 1e-10
    # dense spin operator gives the same answer as the diagonal one
    lo2, hi2, _ = ctx.spin_resolved_wilson(dev(H), 128, 1, dev(np.diag(S).astype(complex)))
    assert phase_dist(lo2.cpu().numpy(), loo) <= PH_TOL
    # uneven split (shape contract only)
    lo3, hi3, _ = ctx.spin_resolved_wilson(dev(H), 128, 1, dev(S), m_lo=60)
    assert lo3.shape == (2, 60) and hi3.shape == (2, 68)   # split inside a PSO cluster: values not unique


def test_config4_full_matrix_size_one_short_loop(ctx):
    """N = 1600, n_occ = 800 -> 2 x 400: 4 loop points (oracle ~10 s)."""
    parts = wl.config4_parts(20)
    H = wl.supercell_grid([parts], 4, 24, t2_indices=[3])
    S = wl.supercell_spin_z(20)
    lo, hi, pso = ctx.spin_resolved_wilson(dev(H), 800, 1, dev(S))
    loo, hio, psoo = wo.spin_resolved_surface(H, 800, 1, S)
    assert np.abs(pso.cpu().numpy() - psoo).max() < 1e-10
    assert phase_dist(lo.cpu().numpy(), loo) <= PH_TOL
    assert phase_dist(hi.cpu().numpy(), hio) <= PH_TOL


# ------------------------------------------------------------------------------ config 5 (reduced)
def test_config5_reduced_wannier_like(ctx):
    p5 = wl.config5_parts()
    H = wl.config5_grid(p5, 64, 64, 65, ix=[0, 17], iy=[3, 31, 60])   # 6 loops x 65 points
    th, ab, mg = ctx.wilson_loop(dev(H), 32, 1)          # [2][3][65][64][64]: batch 2, dims (3, 65)
    tho, abo, mgo = wo.wilson_surface(H, 32, 1)
    assert mgo.min() >= 0.2
    assert phase_dist(th.cpu().numpy(), tho) <= PH_TOL
    # device grid assembly used by bench.py reproduces the host grid
    Ht = wl.config5_grid_torch(p5, 64, 64, 65, "cuda", ix=[0, 17], iy=[3, 31, 60])
    assert np.abs(Ht.cpu().numpy() - H).max() < 1e-12


# ------------------------------------------------------------------------------ host-buffer variants
def test_host_variants_match_device(ctx):
    parts = wl.config4_parts(4, axis="x")
    H = wl.supercell_grid([parts], 6, 5)
    S = wl.supercell_spin_z(4)
    Hh = torch.from_numpy(H).pin_memory()
    ctx.set_workspace_limit(1 << 20)         # force several chunks and the double-buffered stream
    try:
        lo, hi, pso = ctx.spin_resolved_wilson_host(Hh, 32, 1, torch.from_numpy(S))
        th, ab, mg = ctx.wilson_loop_host(Hh, 32, 1)
    finally:
        ctx.set_workspace_limit(110 << 30)
    lod, hid, psod = ctx.spin_resolved_wilson(dev(H), 32, 1, dev(S))
    thd, abd, mgd = ctx.wilson_loop(dev(H), 32, 1)
    # chunking changes the seeded start vectors of the inverse iteration (matrix index inside the
    # chunk), hence the basis inside degenerate subspaces: equal up to rounding, not bitwise
    assert phase_dist(lo.numpy(), lod.cpu().numpy()) < 1e-12 and phase_dist(hi.numpy(), hid.cpu().numpy()) < 1e-12
    assert (pso - psod.cpu()).abs().max() < 1e-12
    assert phase_dist(th.numpy(), thd.cpu().numpy()) < 1e-12 and (mg - mgd.cpu()).abs().max() < 1e-12
    tho, _, _ = wo.wilson_surface(H, 32, 1)
    assert phase_dist(th.numpy(), tho) <= PH_TOL
    # default workspace cap: the host variants still stream the grid in growing chunks (1/8, 1/4, rest)
    th2, _, _ = ctx.wilson_loop_host(Hh, 32, 1)
    assert phase_dist(th2.numpy(), tho) <= PH_TOL
    # loops along the slow grid axis: not contiguous in the host grid (one strided copy per loop)
    th0, _, mg0 = ctx.wilson_loop_host(Hh, 32, 0)
    th0o, _, mg0o = wo.wilson_surface(H, 32, 0)
    assert phase_dist(th0.numpy(), th0o) <= PH_TOL and np.abs(mg0.numpy() - mg0o).max() < 1e-10
    lo0, hi0, _ = ctx.spin_resolved_wilson_host(Hh, 32, 0, torch.from_numpy(S))
    lo0o, hi0o, _ = wo.spin_resolved_surface(H, 32, 0, S)
    assert phase_dist(lo0.numpy(), lo0o) <= PH_TOL and phase_dist(hi0.numpy(), hi0o) <= PH_TOL
    # nested loop on a host grid, with closing phases and a base point
    Hb = wl.config2_grid(14, 12, gamma=0.7)
    Hp, c1, c2 = wl.position_gauge_plane(Hb, np.array([0.11, 0.37, -0.23, 0.41]), np.array([0.29, -0.13, 0.07, 0.33]))
    t1, tn = ctx.nested_wilson_host(torch.from_numpy(Hp[None]).pin_memory(), 2, 1, 0, base=3, wb_lo=1, wb_hi=2,
                                    close1=torch.from_numpy(c1), close2=torch.from_numpy(c2))
    t1o, tno = wo.nested_wilson(Hp, 2, base=3, wb_lo=1, wb_hi=2, close1=c1, close2=c2)
    assert phase_dist(t1.numpy()[0], t1o) <= PH_TOL
    assert wo.circ_sorted_distance(tn.numpy()[0], tno) / (2 * np.pi) <= PH_TOL


def test_only_the_upper_triangle_of_H_is_read(ctx):
    """Header contract: the eigensolver (Jacobi, on-chip, one- and two-stage paths) reads the row-major upper triangle
    only, so the host variants copy just that (N >= 256, 8 row blocks).  NaN in the other triangle must change nothing, on the
    device (one- and two-stage solver) and through the triangle-block host copy, both loop directions."""
    rng = np.random.default_rng(7)
    for N, algo in ((4, 0), (8, 0), (16, 0), (64, 0), (104, 0), (105, 0), (144, 1), (256, 0), (264, 1)):
        A = rng.standard_normal((3, N, N)) + 1j * rng.standard_normal((3, N, N))
        H = (A + A.conj().transpose(0, 2, 1)) / 2
        Hp = H.copy()
        il = np.tril_indices(N, -1)
        Hp[:, il[0], il[1]] = np.nan
        ctx.set_eigh_algorithm(algo)
        try:
            E0, U0 = ctx.eigh_batched(dev(H), N // 2)
            E1, U1 = ctx.eigh_batched(dev(Hp), N // 2)
        finally:
            ctx.set_eigh_algorithm(2)
        assert torch.equal(E0, E1) and torch.equal(U0, U1)
    # host grid, N = 256 (L = 8 supercell), lower triangle poisoned on the host
    parts = wl.config4_parts(8, axis="x")
    H = wl.supercell_grid([parts], 7, 6, t2_indices=[0, 2, 5])
    S = wl.supercell_spin_z(8)
    Hp = H.copy()
    il = np.tril_indices(256, -1)
    Hp[..., il[0], il[1]] = np.nan
    Hh = torch.from_numpy(Hp).pin_memory()
    before = ctx.host_grid_bytes_copied()
    lo, hi, pso = ctx.spin_resolved_wilson_host(Hh, 128, 1, torch.from_numpy(S))
    copied = ctx.host_grid_bytes_copied() - before
    assert copied == H.shape[0] * H.shape[1] * H.shape[2] * sum((256 - r0) * 32 * 16 for r0 in range(0, 256, 32))
    loo, hio, psoo = wo.spin_resolved_surface(H, 128, 1, S)
    assert phase_dist(lo.numpy(), loo) <= PH_TOL and phase_dist(hi.numpy(), hio) <= PH_TOL
    assert np.abs(pso.numpy().reshape(psoo.shape) - psoo).max() < 1e-10
    th0, _, _ = ctx.wilson_loop_host(Hh, 128, 0)            # loops along the slow axis
    th0o, _, _ = wo.wilson_surface(H, 128, 0)
    assert phase_dist(th0.numpy(), th0o) <= PH_TOL


def test_host_grid_streamed_into_one_chunk(ctx):
    """N = 1024 (two-stage eigensolver): the host variant feeds ONE chunk in three sub-ranges (1 + 1 + 2 loops), stage 1
    per sub-range, the rest over the whole batch.  Same phases as the device-resident call and as the oracle (one
    loop), with the unused triangle poisoned on the host."""
    _need_memory(6, ctx)
    parts = wl.config4_parts(16, axis="x")
    H = wl.supercell_grid([parts], 5, 24, t2_indices=[0, 7, 13, 22])
    S = wl.supercell_spin_z(16)
    Hp = H.copy()
    il = np.tril_indices(1024, -1)
    Hp[..., il[0], il[1]] = np.nan
    lo, hi, pso = ctx.spin_resolved_wilson_host(torch.from_numpy(Hp).pin_memory(), 512, 1, torch.from_numpy(S))
    assert ctx.host_schedule() == -3
    lod, hid, psod = ctx.spin_resolved_wilson(dev(H), 512, 1, dev(S))
    assert phase_dist(lo.numpy(), lod.cpu().numpy()) < 1e-10 and phase_dist(hi.numpy(), hid.cpu().numpy()) < 1e-10
    assert (pso - psod.cpu()).abs().max() < 1e-10
    loo, hio, _ = wo.spin_resolved_surface(H[:, 2:3], 512, 1, S)
    assert phase_dist(lo.numpy()[2:3], loo) <= PH_TOL and phase_dist(hi.numpy()[2:3], hio) <= PH_TOL
    th, _, mg = ctx.wilson_loop_host(torch.from_numpy(Hp).pin_memory(), 512, 1)
    thd, _, mgd = ctx.wilson_loop(dev(H), 512, 1)
    assert phase_dist(th.numpy(), thd.cpu().numpy()) < 1e-10 and (mg - mgd.cpu()).abs().max() < 1e-10


def test_chunk_pipeline_matches_single_chunk_and_oracle(ctx):
    """A small workspace cap splits the loops into >= 3 chunks: the two-stream chunk pipeline
    (tridiagonalization of chunk c+1 next to the rest of chunk c, two scratch regions) must give
    the results of the single-chunk run (to rounding: the start vectors of inverse iteration are
    seeded by the index inside the chunk) and match the oracle."""
    parts = wl.config3_parts(2, L=4)                       # N = 64
    H = wl.supercell_grid([parts], 9, 5)                   # 5 loops of 9 points
    Hd = dev(H)
    th1, ab1, mg1 = ctx.wilson_loop(Hd, 32, 1)
    S = wl.supercell_spin_z(4)
    lo1, hi1, pso1 = ctx.spin_resolved_wilson(Hd, 32, 1, dev(S))
    try:
        ctx.set_workspace_limit(5 << 20)                   # one loop per chunk -> 5 chunks
        ctx.set_chunk_pipeline(True)
        th2, ab2, mg2 = ctx.wilson_loop(Hd, 32, 1)
        lo2, hi2, pso2 = ctx.spin_resolved_wilson(Hd, 32, 1, dev(S))
        torch.cuda.synchronize()
    finally:
        ctx.set_workspace_limit(64 << 30)
        ctx.set_chunk_pipeline(False)
    assert phase_dist(th1.cpu().numpy(), th2.cpu().numpy()) <= 1e-11
    assert (mg1 - mg2).abs().max().item() <= 1e-12 and (pso1 - pso2).abs().max().item() <= 1e-12
    assert phase_dist(lo1.cpu().numpy(), lo2.cpu().numpy()) <= 1e-11
    assert phase_dist(hi1.cpu().numpy(), hi2.cpu().numpy()) <= 1e-11
    tho, _, _ = wo.wilson_surface(H, 32, 1)
    assert phase_dist(th2.cpu().numpy(), tho) <= PH_TOL
    loo, hio, _ = wo.spin_resolved_surface(H, 32, 1, S)
    assert phase_dist(lo2.cpu().numpy(), loo) <= PH_TOL and phase_dist(hi2.cpu().numpy(), hio) <= PH_TOL


# ------------------------------------------------------------------------------ full sizes, bench configuration
def _bench_workload(cfg):
    import importlib.util, os
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(os.path.dirname(__file__), "..", "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod.Workload(cfg, 0, False)


def _need_memory(gb, ctx=None):
    if ctx is not None:
        ctx.release_workspace()          # the arena of an earlier large call stays allocated otherwise
        torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < gb * 2 ** 30:
        pytest.skip(f"needs {gb} GB of free device memory")


def test_full_size_config4_in_bench_configuration(ctx):
    """BASELINE.json configs[3] at full size exactly as bench.py runs it (N = 1600, 24 x 25 grid, default
    workspace cap and eigensolver selection: the two-stage reduction for N = 1600, the one-stage one for the
    PSO): exact invariants on the whole output, and four sampled loops element by element against the
    oracle (one loop of 25 k-points costs the oracle ~15 s)."""
    _need_memory(30, ctx)
    wk = _bench_workload(4)
    H, S = wk.device_grid(torch, torch.device("cuda"))
    lo, hi, pso = wk.run_device(ctx, H, S)
    torch.cuda.synchronize()
    # PSO eigenvalues are exactly +-1 ([H, S_z] = 0), half of each sign
    p = pso.cpu().numpy()
    assert np.abs(np.abs(p) - 1.0).max() < 1e-10 and np.all(p[..., :400] < 0) and np.all(p[..., 400:] > 0)
    # sector windings over the closed t2 cycle: +1 (S_z = -1 sector), -1, total 0 -- exact integers (R11)
    wl_lo = ctx.winding(lo[None]).item()
    wl_hi = ctx.winding(hi[None]).item()
    assert abs(wl_lo - round(wl_lo)) < 1e-9 and abs(wl_hi - round(wl_hi)) < 1e-9
    assert sorted((round(wl_lo), round(wl_hi))) == [-1, 1]
    parts = wl.config4_parts(20, realization=0)
    Sh = wl.supercell_spin_z(20)
    for j in (0, 5, 11, 17):
        Hj = H[0, j].cpu().numpy()[None, None]                          # the same matrices on both sides
        assert np.abs(wl.supercell_grid([parts], 25, 24, t2_indices=[j]) - Hj).max() < 1e-12   # = the seeded recipe
        loo, hio, _ = wo.spin_resolved_surface(Hj, 800, 1, Sh)
        assert phase_dist(lo[j:j + 1].cpu().numpy(), loo) <= PH_TOL
        assert phase_dist(hi[j:j + 1].cpu().numpy(), hio) <= PH_TOL
    del H
    torch.cuda.empty_cache()


def test_full_size_config4_spin_mixing_variant_one_loop(ctx):
    """SURVEY 8(d), config 4 "second, harder variant for tests": impurity fields along x do not commute with
    S_z, the PSO eigenvalues leave +-1 and its 800 eigenvectors are non-degenerate -- one whole
    loop (25 k-points) at N = 1600 / m = 800 against the oracle, element by element."""
    _need_memory(12, ctx)
    parts = wl.config4_parts(20, axis="x")
    H = wl.supercell_grid([parts], 25, 24, t2_indices=[7])
    S = wl.supercell_spin_z(20)
    lo, hi, pso = ctx.spin_resolved_wilson(dev(H), 800, 1, dev(S))
    loo, hio, psoo = wo.spin_resolved_surface(H, 800, 1, S)
    assert np.abs(np.abs(psoo) - 1).max() > 1e-3 and np.abs(psoo).min() > 0.5     # spin mixing, still gapped at 400 | 400
    assert np.abs(pso.cpu().numpy() - psoo).max() < 1e-10
    assert phase_dist(lo.cpu().numpy(), loo) <= PH_TOL
    assert phase_dist(hi.cpu().numpy(), hio) <= PH_TOL


def test_full_size_config3_sampled(ctx):
    """BASELINE.json configs[2] at full size (16 realizations x 32 x 33, N = 400; 43 GB): 32 sampled loops
    against the oracle, sum rule sum_n theta_n = arg det W on all loops is implied by the eigen-solver
    parity; total winding per realization is an exact integer (0: time-reversal symmetric)."""
    _need_memory(50, ctx)
    wk = _bench_workload(3)
    H, _ = wk.device_grid(torch, torch.device("cuda"))
    th, ab, mg = wk.run_device(ctx, H, None)
    torch.cuda.synchronize()
    assert mg.min().item() > 0.5
    w = ctx.winding(th.reshape(16, 32, 200)).cpu().numpy()
    assert np.abs(w - np.round(w)).max() < 1e-8 and np.all(np.round(w) == 0)
    for (r, j) in [(r, j) for r in (0, 5, 10, 15) for j in (0, 3, 9, 13, 18, 22, 27, 31)]:   # 32 loops, 4 realizations
        Hl = H[r, j].cpu().numpy()[None, None]
        tho, abo, mgo = wo.wilson_surface(Hl, 200, 1)
        assert phase_dist(th[r * 32 + j:r * 32 + j + 1].cpu().numpy(), tho) <= PH_TOL
        assert abs(mg[r * 32 + j].item() - mgo[0]) < 1e-9
    del H
    torch.cuda.empty_cache()


def test_full_size_config5_sampled(ctx):
    """BASELINE.json configs[4] at full size (64 x 64 loops of 65 points, N = 64: 266 240 eigensolves)."""
    _need_memory(25, ctx)
    wk = _bench_workload(5)
    H, _ = wk.device_grid(torch, torch.device("cuda"))
    th, ab, mg = wk.run_device(ctx, H, None)
    torch.cuda.synchronize()
    assert mg.min().item() > 0.2                               # harness asserts the gap (R13)
    idx = list(range(0, 4096, 16)) + [77, 1234, 4095]     # 259 of the 4096 loops
    for l in idx:
        Hl = H[l // 64, l % 64].cpu().numpy()[None, None]
        tho, abo, _ = wo.wilson_surface(Hl, 32, 1)
        assert phase_dist(th[l:l + 1].cpu().numpy(), tho) <= PH_TOL
    del H
    torch.cuda.empty_cache()


def test_assemble_bloch_matches_the_input_recipe(ctx):
    """NEXT-1: H_grid assembled on the device as one GEMM reproduces the seeded generators."""
    # twisted supercell (config 3 pieces, L = 4): blocks [H_bulk, Bx, Bx^dagger, By, By^dagger]
    Hb, Bx, By = wl.config3_parts(3, L=4)
    A = np.stack([Hb, Bx, Bx.conj().T, By, By.conj().T])
    R = [[0, 0], [1, 0], [-1, 0], [0, 1], [0, -1]]
    n1, n2 = 9, 5
    t = np.array([[i / n1, j / n2] for j in range(n2) for i in range(n1)])
    H = ctx.assemble_bloch(dev(A), dev(t), R).cpu().numpy().reshape(n2, n1, 64, 64)
    Href = wl.supercell_grid([(Hb, Bx, By)], n1, n2)[0]
    assert np.abs(H - Href).max() < 1e-13
    # config 5: on-site block + 13 half-space vectors and their conjugates
    H0, Rs, HR = wl.config5_parts()
    A = np.concatenate([H0[None], HR, HR.conj().transpose(0, 2, 1)])
    R = [[0, 0, 0]] + [list(map(int, r)) for r in Rs] + [list(map(int, -r)) for r in Rs]
    rng = np.random.default_rng(1)
    t = rng.uniform(0, 1, (37, 3))
    H = ctx.assemble_bloch(dev(A), dev(t), R).cpu().numpy()
    for k in (0, 17, 36):
        assert np.abs(H[k] - wl.assemble_config5((H0, Rs, HR), 2 * np.pi * t[k])).max() < 1e-12
    assert np.abs(H - H.conj().transpose(0, 2, 1)).max() < 1e-13


def test_plaquette_flux_matches_oracle(ctx):
    """NEXT-2: plaquette Berry fluxes (coupling-matrix method), plain and spin resolved."""
    G = wl.qwz_grid(20, 20)                                            # Eq. 4, m = 1
    f = ctx.plaquette_flux(dev(G[None]), 1).cpu().numpy()[0]
    fo = wo.plaquette_flux(G, 1)
    assert np.abs(wo.wrap_pi(f - fo)).max() <= PH_TOL * 2 * np.pi
    assert round(f.sum() / (2 * np.pi)) == 1                           # C = 1
    H = wl.config1_grid(16, 12)                                        # BHZ, m = 2 -> sectors 1 + 1
    f = ctx.plaquette_flux(dev(H[None]), 2).cpu().numpy()[0]
    assert np.abs(wo.wrap_pi(f - wo.plaquette_flux(H, 2))).max() <= PH_TOL * 2 * np.pi
    flo, fhi, pso = ctx.plaquette_flux(dev(H[None]), 2, dev(wl.bhz4_spin_z()), want_pso=True)
    floo, fhio = wo.plaquette_flux(H, 2, wl.bhz4_spin_z())
    assert np.abs(wo.wrap_pi(flo.cpu().numpy()[0] - floo)).max() <= PH_TOL * 2 * np.pi
    assert np.abs(wo.wrap_pi(fhi.cpu().numpy()[0] - fhio)).max() <= PH_TOL * 2 * np.pi
    assert (round(flo.sum().item() / (2 * np.pi)), round(fhi.sum().item() / (2 * np.pi))) == (-1, 1)
    assert np.abs(np.abs(pso.cpu().numpy()) - 1).max() < 1e-12
    # disordered supercell, two realizations in the batch, ragged grid, tridiagonalization path + LU of 32 x 32
    parts = [wl.config3_parts(r, L=4) for r in (0, 1)]
    Hs = wl.supercell_grid(parts, 5, 4)                                # [2][4][5][64][64]
    f = ctx.plaquette_flux(dev(Hs), 32).cpu().numpy()
    for r in range(2):
        assert np.abs(wo.wrap_pi(f[r] - wo.plaquette_flux(Hs[r], 32))).max() <= PH_TOL * 2 * np.pi
    S = wl.supercell_spin_z(4)
    flo, fhi = ctx.plaquette_flux(dev(Hs), 32, dev(S))
    floo, fhio = wo.plaquette_flux(Hs[1], 32, S)
    assert np.abs(wo.wrap_pi(flo.cpu().numpy()[1] - floo)).max() <= PH_TOL * 2 * np.pi
    assert np.abs(wo.wrap_pi(fhi.cpu().numpy()[1] - fhio)).max() <= PH_TOL * 2 * np.pi


def test_chiral_hoti_eq9_on_device(ctx):
    """NEXT-4: the paper's second worked example (Eq. 9) through the C ABI: nested loops for 20 k_z slices
    in one batched call, spin-resolved surface at k_z = 0; invariants exact, phases against the oracle."""
    kzs = [j / 20 for j in range(20)]
    Hz = wl.chiral_hoti_grid(24, 24, kzs, 1.0)                              # [20][24][24][4][4]
    th1, thn = ctx.nested_wilson(dev(Hz), 2, 1, 0)                          # batch = k_z
    thn = thn.cpu().numpy()
    for a in (0, 3, 11, 19):
        th1o, thno = wo.nested_wilson(Hz[a], 2)
        assert phase_dist(th1.cpu().numpy()[a], th1o) <= PH_TOL
        assert wo.circ_sorted_distance(thn[a], thno) / (2 * np.pi) <= PH_TOL
    w = ctx.winding(dev(thn[None])).item()
    assert abs(w - round(w)) < 1e-9 and abs(round(w)) == 1                   # gapless nested spectrum
    H = wl.chiral_hoti_grid(32, 32, [0.0], 1.0)
    S = wl.chiral_hoti_spin()
    lo, hi, pso = ctx.spin_resolved_wilson(dev(H), 2, 1, dev(S))
    loo, hio, psoo = wo.spin_resolved_surface(H, 2, 1, S)
    assert phase_dist(lo.cpu().numpy(), loo) <= PH_TOL and phase_dist(hi.cpu().numpy(), hio) <= PH_TOL
    assert np.abs(pso.cpu().numpy() - psoo).max() < 1e-12
    wlo, whi = ctx.winding(lo[None]).item(), ctx.winding(hi[None]).item()
    assert sorted((round(wlo), round(whi))) == [-1, 1]                       # |C_s| = 1


def test_fused_bloch_generation_matches_materialised_grid(ctx):
    """NEXT-1 fused in front of S1: loops on a grid that is generated chunk by chunk from real-space blocks
    equal the loops on the materialised H_grid (same seeded recipe), and the oracle."""
    # two disorder realizations of the twisted 6 x 6 supercell (N = 144: blocked path), grid 3 x 9
    parts = [wl.config3_parts(r, L=6) for r in (0, 1)]
    A = np.stack([np.stack([Hb, Bx, Bx.conj().T, By, By.conj().T]) for (Hb, Bx, By) in parts])   # [2][5][N][N]
    R = [[0, 0], [0, 1], [0, -1], [1, 0], [-1, 0]]            # grid axes (t2, t1): Bx goes with the t1 axis
    H = wl.supercell_grid(parts, 9, 3)                          # [2][3][9][144][144]
    th, ab, mg = ctx.wilson_loop(dev(H), 72, 1)
    try:
        ctx.set_workspace_limit(40 << 20)                       # several chunks, chunks spanning realizations
        thb, abb, mgb = ctx.wilson_loop_bloch(dev(A), R, (3, 9), 72, 1)
        S = wl.supercell_spin_z(6)
        lob, hib, psob = ctx.spin_resolved_wilson_bloch(dev(A), R, (3, 9), 72, 1, dev(S))
        torch.cuda.synchronize()
    finally:
        ctx.set_workspace_limit(64 << 30)
    assert phase_dist(thb.cpu().numpy(), th.cpu().numpy()) <= 1e-10
    assert (mgb - mg).abs().max().item() < 1e-11
    tho, _, _ = wo.wilson_surface(H, 72, 1)
    assert phase_dist(thb.cpu().numpy(), tho) <= PH_TOL
    loo, hio, _ = wo.spin_resolved_surface(H, 72, 1, S)
    assert phase_dist(lob.cpu().numpy(), loo) <= PH_TOL and phase_dist(hib.cpu().numpy(), hio) <= PH_TOL
    # small matrices (Jacobi path): config 1 from its three hopping blocks
    T0 = np.kron(wl.sz, wl.s0).astype(complex)                                   # on-site m = 1
    Tx = np.kron(wl.sx, wl.sz) / 2j - np.kron(wl.sz, wl.s0) / 2
    Ty = np.kron(wl.sy, wl.s0) / 2j - np.kron(wl.sz, wl.s0) / 2
    A1 = np.stack([T0, Tx, Tx.conj().T, Ty, Ty.conj().T])[None]
    R1 = [[0, 0], [0, 1], [0, -1], [1, 0], [-1, 0]]                              # axes (ky, kx)
    H1 = wl.config1_grid(20, 11)
    th1, _, _ = ctx.wilson_loop_bloch(dev(A1), R1, (11, 20), 2, 1)
    th1o, _, _ = wo.wilson_surface(H1[None], 2, 1)
    assert phase_dist(th1.cpu().numpy(), th1o) <= PH_TOL
    # on-chip path (N = 64): config 5 blocks, loops along kz
    H0, Rs, HR = wl.config5_parts()
    A5 = np.concatenate([H0[None], HR, HR.conj().transpose(0, 2, 1)])[None]
    R5 = [[0, 0, 0]] + [list(map(int, r)) for r in Rs] + [list(map(int, -r)) for r in Rs]
    th5, _, _ = ctx.wilson_loop_bloch(dev(A5), R5, (2, 3, 13), 32, 2)
    H5 = np.array([[[wl.assemble_config5((H0, Rs, HR), 2 * np.pi * np.array([i / 2, j / 3, l / 13])) for l in range(13)]
                    for j in range(3)] for i in range(2)])
    th5o, _, _ = wo.wilson_surface(H5[None], 32, 2)
    assert phase_dist(th5.cpu().numpy(), th5o) <= PH_TOL


def test_band_windows_match_oracle(ctx):
    """NEXT-3: be_wilson_loop_window / be_spin_resolved_wilson_window on the Jacobi, on-chip and blocked
    eigensolver paths: phases, both-edge gap flag, the paper's upper-band Chern number, completeness."""
    from paper_2312_13051_b200.binding import BerryEasyError
    # Eq. 4, upper band: C = -1
    H = wl.qwz_grid(40, 40)[None]
    th, ab, mg = ctx.wilson_loop(dev(H), 2, 1, band_lo=1)
    tho, abo, mgo = wo.wilson_surface_window(H, 1, 2, 1)
    assert phase_dist(th.cpu().numpy(), tho) <= PH_TOL
    assert np.abs(mg.cpu().numpy() - mgo).max() < 1e-12
    assert wo.chern_number(th.cpu().numpy()) == -1
    # BHZ: unoccupied pair; all four bands (W = 1, no inner edge); the degenerate middle window is flagged
    Hb = wl.config1_grid(30, 7)[None]
    th, ab, mg = ctx.wilson_loop(dev(Hb), 4, 1, band_lo=2)
    tho, abo, mgo = wo.wilson_surface_window(Hb, 2, 4, 1)
    assert phase_dist(th.cpu().numpy(), tho) <= PH_TOL and np.abs(mg.cpu().numpy() - mgo).max() < 1e-12
    th, ab, mg = ctx.wilson_loop(dev(Hb), 4, 1, band_lo=0)
    assert np.abs(th.cpu().numpy()).max() < 1e-10 and np.all(np.isinf(mg.cpu().numpy()))
    _, _, mg = ctx.wilson_loop(dev(Hb), 3, 1, band_lo=1)
    assert mg.cpu().numpy().max() < 1e-10
    S = wl.bhz4_spin_z()
    lo, hi, pso = ctx.spin_resolved_wilson_window(dev(Hb), 2, 4, 1, dev(S))
    loo, hio, psoo = wo.spin_resolved_surface(Hb, 4, 1, S, band_lo=2)
    assert phase_dist(lo.cpu().numpy(), loo) <= PH_TOL and phase_dist(hi.cpu().numpy(), hio) <= PH_TOL
    assert np.abs(pso.cpu().numpy() - psoo).max() < 1e-10
    # on-chip path (N = 64): a window across the gap
    p5 = wl.config5_parts()
    H5 = wl.config5_grid(p5, 64, 64, 13, ix=[3], iy=[5, 40])
    th, ab, mg = ctx.wilson_loop(dev(H5), 40, 1, band_lo=24)      # [1][2][13][64][64]: batch 1, dims (2, 13)
    tho, abo, mgo = wo.wilson_surface_window(H5, 24, 40, 1)
    assert mgo.min() > 1e-4
    assert phase_dist(th.cpu().numpy(), tho) <= PH_TOL and np.abs(mg.cpu().numpy() - mgo).max() < 1e-10
    # blocked path: the same recipe with 56 spatial orbitals (N = 112), window [40, 70) across the gap.  (A
    # window edge inside the DISORDERED bands of config 3 is no parity case: the oracle's own phases move by
    # 0.4 rad under a 1e-12 perturbation there, |lambda| down to 1e-16.)
    p7 = wl.config5_parts(norb_spatial=56)
    H7 = wl.config5_grid(p7, 64, 64, 17, ix=[3], iy=[5, 40])
    th, ab, mg = ctx.wilson_loop(dev(H7), 70, 1, band_lo=40)
    tho, abo, mgo = wo.wilson_surface_window(H7, 40, 70, 1)
    assert mgo.min() > 1e-2 and np.abs(mg.cpu().numpy() - mgo).max() < 1e-10
    assert phase_dist(th.cpu().numpy(), tho) <= PH_TOL
    with pytest.raises(BerryEasyError):
        ctx.wilson_loop(dev(Hb), 2, 1, band_lo=2)      # empty window
    with pytest.raises(BerryEasyError):
        ctx.wilson_loop(dev(Hb), 5, 1, band_lo=1)      # band_hi > N


def test_launch_counter_counts_kernels(ctx):
    n0 = ctx.launch_count()
    ctx.wilson_loop(dev(wl.config1_grid(6, 2)[None]), 2, 1)
    assert ctx.launch_count() > n0


# ------------------------------------------------------------------------------ S2/S3 building block
@pytest.mark.parametrize("opA,opB", [("N", "N"), ("N", "C"), ("C", "N"), ("N", "T"), ("T", "N"), ("J", "N"),
                                     ("N", "J"), ("C", "C"), ("T", "J")])
def test_zgemm_batched_op_pairs_ragged_against_plain_matmul(ctx, opA, opB):
    """be_zgemm_batched = alpha op(A) op(B) + beta C (the contraction of Eq. 2's links and of the ordered
    product) against numpy's matmul, on sizes that span several 64 x 32 x 16 tiles with
    ragged tails in M, N and K, with padding in the leading dimensions."""
    rng = np.random.default_rng(7)
    op = {"N": lambda X: X, "T": lambda X: X.transpose(0, 2, 1), "C": lambda X: X.conj().transpose(0, 2, 1),
          "J": lambda X: X.conj()}
    for (M, N, K, batch) in [(150, 77, 45, 3), (64, 32, 16, 2), (1, 1, 1, 1), (70, 33, 130, 2)]:
        shA = (K, M) if opA in "TC" else (M, K)
        shB = (N, K) if opB in "TC" else (K, N)
        A = rng.standard_normal((batch,) + shA) + 1j * rng.standard_normal((batch,) + shA)
        B = rng.standard_normal((batch,) + shB) + 1j * rng.standard_normal((batch,) + shB)
        C0 = rng.standard_normal((batch, M, N)) + 1j * rng.standard_normal((batch, M, N))
        alpha, beta = 0.7 - 0.3j, -0.2 + 1.1j
        want = alpha * (op[opA](A) @ op[opB](B)) + beta * C0
        # column-major storage with padded leading dimensions: X[b] is stored as its transpose, row-major
        def colmajor(X, pad):
            b, r, c = X.shape
            buf = np.zeros((b, c, r + pad), dtype=np.complex128)
            buf[:, :, :r] = X.transpose(0, 2, 1)
            return buf
        Ad, Bd, Cd = dev(colmajor(A, 3)), dev(colmajor(B, 1)), dev(colmajor(C0, 2))
        lda, ldb, ldc = shA[0] + 3, shB[0] + 1, M + 2
        ctx.zgemm_batched(opA, opB, Ad, Bd, Cd, M, N, K, lda, ldb, ldc, shA[1] * lda, shB[1] * ldb, N * ldc, batch,
                          alpha=alpha, beta=beta)
        torch.cuda.synchronize()
        got = Cd.cpu().numpy()[:, :, :M].transpose(0, 2, 1)
        scale = np.abs(A).max() * np.abs(B).max() * K + np.abs(C0).max()
        assert np.abs(got - want).max() <= 1e-14 * scale * 4, (opA, opB, M, N, K)
        assert np.all(Cd.cpu().numpy()[:, :, M:] == 0)     # the padding rows are never written


def test_zgemm_lower_touches_only_tiles_on_or_below_the_diagonal(ctx):
    rng = np.random.default_rng(8)
    n, k, batch = 200, 64, 2
    V = rng.standard_normal((batch, n, k)) + 1j * rng.standard_normal((batch, n, k))
    C0 = rng.standard_normal((batch, n, n)) + 1j * rng.standard_normal((batch, n, n))
    Vd = dev(V.transpose(0, 2, 1))          # column-major [n][k]
    Cd = dev(C0.transpose(0, 2, 1))
    ctx.zgemm_batched("N", "C", Vd, Vd, Cd, n, n, k, n, n, n, n * k, n * k, n * n, batch, alpha=-1.0 + 0j, beta=1.0 + 0j,
                      lower=True)
    torch.cuda.synchronize()
    got = Cd.cpu().numpy().transpose(0, 2, 1)
    want = C0 - V @ V.conj().transpose(0, 2, 1)
    low = np.tril(np.ones((n, n), dtype=bool))
    assert np.abs(got - want)[:, low].max() <= 1e-12
    # strictly above the 64 x 32 tile staircase nothing was written
    r, c = np.indices((n, n))
    untouched = (c // 32) > (2 * (r // 64) + 1)
    assert np.all(got[:, untouched] == C0[:, untouched])
