"""Pins for oracle/wilson_oracle.py against what the paper and the mathematics fix.

None of these tests re-types the oracle's formulas: each compares it with a printed value
(tests/golden/paper_pins.txt), a closed form, an invariant, an exact identity or a brute-force
evaluation that takes a different route.  All run on CPU (``-m "not gpu"``).
"""
import os

import numpy as np
import pytest

from oracle import wilson_oracle as wo
from paper_2312_13051_b200 import workloads as wl

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    out = {}
    with open(os.path.join(HERE, "golden", "paper_pins.txt")) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if "=" in line:
                k, v = line.split("=", 1)
                out[k.strip()] = float(v)
    return out


GOLD = _golden()


# ------------------------------------------------------------------ closed-form helpers (test side)
def lower_band_vector(d):
    """Closed-form lower eigenvector of d.sigma (E = -|d|), gauge irrelevant."""
    dx, dy, dz = d
    n = np.sqrt(dx * dx + dy * dy + dz * dz)
    if dz <= 0:
        v = np.array([dz - n, dx + 1j * dy])
    else:  # avoid the cancellation / zero vector at d = (0,0,+|d|)
        v = np.array([-(dx - 1j * dy), dz + n])
    return v / np.linalg.norm(v)


def qwz_d(kx, ky, M=1.5):
    return np.array([np.sin(kx), np.sin(ky), np.cos(kx) + np.cos(ky) + M])


# ------------------------------------------------------------------ SSH
def test_ssh_berry_phase_quantized():
    H, _ = wl.ssh_loop(1.0, 0.5, 50)
    th, ab, _ = wo.wilson_loop(H, 1)
    assert abs(wo.wrap_pi(th[0] - np.pi * GOLD["ssh_trivial_phase_over_pi"])) < 1e-12
    H, _ = wl.ssh_loop(0.5, 1.0, 50)
    th, ab, _ = wo.wilson_loop(H, 1)
    assert abs(wo.wrap_pi(th[0] - np.pi * GOLD["ssh_topological_phase_over_pi"])) < 1e-12
    # both bands: total phase = arg det W = 0 or 2 pi * integer, and the upper band mirrors it
    th2, _, _ = wo.wilson_loop(H, 2)
    assert abs(wo.wrap_pi(np.sum(th2))) < 1e-10


def test_ssh_position_gauge_needs_closing_phase():
    """R6: in the position gauge (r_B = 1/2) the loop phase is the periodic-gauge one shifted by
    -2 pi * <r> = -pi/2 (chiral symmetry puts weight exactly 1/2 on sublattice B); without the
    closing phase Phi the two dimerizations become indistinguishable."""
    for (v, w), per in (((1.0, 0.5), 0.0), ((0.5, 1.0), np.pi)):
        H, phi = wl.ssh_loop(v, w, 50, position_gauge=True)
        th, _, _ = wo.wilson_loop(H, 1, close=phi)
        assert abs(wo.wrap_pi(th[0] - (per - np.pi / 2))) < 1e-12
    Ha, phi = wl.ssh_loop(1.0, 0.5, 50, position_gauge=True)
    Hb, _ = wl.ssh_loop(0.5, 1.0, 50, position_gauge=True)
    ta, _, _ = wo.wilson_loop(Ha, 1)
    tb, _, _ = wo.wilson_loop(Hb, 1)
    assert abs(wo.wrap_pi(ta[0] - tb[0])) < 1e-10  # a missing Phi is caught by the test above


# ------------------------------------------------------------------ QWZ Eq. 4
def test_qwz_chern_number_is_one_paper_value():
    H = wl.qwz_grid(100, 100)
    th, ab, mg = wo.wilson_surface(H[None], 1, direction=1)
    assert wo.chern_number(th) == int(GOLD["qwz_eq4_chern"])
    assert abs(-wo.winding(th) - 1.0) < 1e-12
    assert mg.min() > 0.9
    # trivial phase of the same model: M = 2.5 -> C = 0
    th0, _, _ = wo.wilson_surface(wl.qwz_grid(40, 40, M=2.5)[None], 1, direction=1)
    assert wo.chern_number(th0) == 0


def test_band_windows_upper_band_completeness_and_edge_gaps():
    """NEXT-3 band windows [lo, hi) (PAPER.md:79 ``bands``): (i) the Chern numbers of all bands sum to
    zero, so Eq. 4's upper band carries -C of the printed lower-band value; (ii) its loops equal the
    scalar products of the closed-form upper eigenvectors; (iii) the window of ALL bands has W = 1
    (completeness of the eigenbasis, periodic gauge); (iv) the gap flag looks at both window edges."""
    H = wl.qwz_grid(60, 60)
    th_up, _, mg = wo.wilson_surface_window(H[None], 1, 2, direction=1)
    assert wo.chern_number(th_up) == -int(GOLD["qwz_eq4_chern"])
    assert mg.min() > 0.9
    n1 = 60
    for i2 in (0, 7, 31):
        ky = 2 * np.pi * i2 / 60
        vecs = [lower_band_vector(-qwz_d(2 * np.pi * j / n1, ky)) for j in range(n1)]   # upper band of d.sigma
        w = 1.0 + 0j
        for j in range(n1):
            w *= np.vdot(vecs[j], vecs[(j + 1) % n1])
        assert abs(np.angle(np.exp(1j * (th_up[i2, 0] - np.angle(w))))) < 1e-12
    Hb = wl.config1_grid(12, 5)[None]
    th_all, ab_all, mg_all = wo.wilson_surface_window(Hb, 0, 4, direction=1)
    assert np.abs(th_all).max() < 1e-12 and np.abs(ab_all - 1).max() < 1e-12
    assert np.all(np.isinf(mg_all))                       # no edge inside the spectrum
    th_lo, _, mg_lo = wo.wilson_surface_window(Hb, 0, 2, direction=1)
    th_ref, _, mg_ref = wo.wilson_surface(Hb, 2, direction=1)
    assert np.array_equal(th_lo, th_ref) and np.array_equal(mg_lo, mg_ref)
    _, _, mg_mid = wo.wilson_surface_window(Hb, 1, 3, direction=1)
    assert mg_mid.max() < 1e-12                           # BHZ bands are two-fold degenerate: both edges closed


def test_qwz_chern_matches_berry_curvature_plaquette_sum():
    """Independent route (Eq. 5, PAPER.md:69 with A = i<u|d_k u>, Eq. 1): lattice field strength
    from closed-form eigenvectors, summed over plaquettes.  <u_k|u_{k+dk}> ~ 1 - i A dk, so the
    counter-clockwise plaquette flux is -arg(prod of links)."""
    n = 40
    ks = 2 * np.pi * np.arange(n) / n
    u = [[lower_band_vector(qwz_d(kx, ky)) for ky in ks] for kx in ks]
    tot = 0.0
    for i in range(n):
        for j in range(n):
            a, b = u[i][j], u[(i + 1) % n][j]
            c, d = u[(i + 1) % n][(j + 1) % n], u[i][(j + 1) % n]
            tot += -np.angle(np.vdot(a, b) * np.vdot(b, c) * np.vdot(c, d) * np.vdot(d, a))
    C_curv = tot / (2 * np.pi)
    assert abs(C_curv - round(C_curv)) < 1e-10
    # Stokes with F_xy = d_x A_y - d_y A_x and a gauge periodic along the loop direction:
    #   int F = -int dky d_ky (oint dkx A_x)  =>  flow of xbar_x(ky) (Eq. 6) = -C_curvature,
    #   int F = +int dkx d_kx (oint dky A_y)  =>  flow of xbar_y(kx)         = +C_curvature.
    # The paper quotes C = 1 from the kx-loop flow; Eq. 5 read literally has the
    # opposite orientation (reading R15).  Both orientations are pinned here.
    G = wl.qwz_grid(n, n)[None]
    th, _, _ = wo.wilson_surface(G, 1, direction=1)   # loops along kx, flow in ky
    assert wo.chern_number(th) == -int(round(C_curv)) == int(GOLD["qwz_eq4_chern"])
    th, _, _ = wo.wilson_surface(G, 1, direction=0)   # loops along ky, flow in kx
    assert wo.chern_number(th) == int(round(C_curv))


def test_plaquette_flux_chern_number_and_stokes():
    """NEXT-2: plaquette fluxes.  Pins: (i) Eq. 4: sum of the fluxes / 2 pi = C = 1
    (PAPER.md:67, 91); (ii) closed-form lower-band vectors give the same flux plaquette by plaquette;
    (iii) Stokes on a row of plaquettes, exact at finite grids because det is Abelian:
    sum_i flux[j][i] = Theta_j - Theta_{j+1} (mod 2 pi) with Theta = sum_n theta_n of the kx loops;
    (iv) BHZ: sector Chern numbers -1 / +1 = -winding (R3), total 0."""
    n = 20
    G = wl.qwz_grid(n, n)
    f = wo.plaquette_flux(G, 1)
    assert abs(f.sum() / (2 * np.pi) - int(GOLD["qwz_eq4_chern"])) < 1e-12
    ks = 2 * np.pi * np.arange(n) / n
    u = [[lower_band_vector(qwz_d(kx, ky)) for kx in ks] for ky in ks]        # [ky][kx]
    for (j, i) in ((0, 0), (3, 17), (19, 19)):
        a, b = u[j][i], u[j][(i + 1) % n]
        c, d = u[(j + 1) % n][(i + 1) % n], u[(j + 1) % n][i]
        ref = np.angle(np.vdot(a, b) * np.vdot(b, c) * np.vdot(c, d) * np.vdot(d, a))
        assert abs(wo.wrap_pi(f[j, i] - ref)) < 1e-12
    th, _, _ = wo.wilson_surface(G[None], 1, 1)
    Th = th.sum(1)
    assert np.abs(wo.wrap_pi(f.sum(1) - (Th - np.roll(Th, -1)))).max() < 1e-12
    H = wl.config1_grid(16, 12)
    th, _, _ = wo.wilson_surface(H[None], 2, 1)
    Th = th.sum(1)
    assert np.abs(wo.wrap_pi(wo.plaquette_flux(H, 2).sum(1) - (Th - np.roll(Th, -1)))).max() < 1e-12
    flo, fhi = wo.plaquette_flux(H, 2, wl.bhz4_spin_z())
    clo, chi = flo.sum() / (2 * np.pi), fhi.sum() / (2 * np.pi)
    assert abs(clo + 1) < 1e-12 and abs(chi - 1) < 1e-12
    lo, hi, _ = wo.spin_resolved_surface(H[None], 2, 1, wl.bhz4_spin_z())
    assert wo.chern_number(lo) == round(clo) and wo.chern_number(hi) == round(chi)


def test_abelian_loop_equals_scalar_product_of_closed_form_vectors():
    """m = 1: W = prod_j <u_j|u_{j+1}> is a scalar; u from the closed form, not from eigh."""
    n1 = 37
    for ky in (0.3, 2.1, 4.0):
        Hl = np.array([wl.qwz_eq4(2 * np.pi * i / n1, ky) for i in range(n1)])
        us = [lower_band_vector(qwz_d(2 * np.pi * i / n1, ky)) for i in range(n1)]
        Wb = 1.0 + 0j
        for j in range(n1):
            Wb *= np.vdot(us[j], us[(j + 1) % n1])
        th, ab, _ = wo.wilson_loop(Hl, 1)
        assert abs(wo.wrap_pi(th[0] - np.angle(Wb))) < 1e-12
        assert abs(ab[0] - abs(Wb)) < 1e-12


def test_wilson_matrix_brute_force_index_loops():
    """4x4 model, m = 2: the ordered product written out with explicit index sums, and
    sum theta = arg det W = sum_j arg det M_j (mod 2 pi)."""
    n1 = 9
    Hl = np.array([wl.bhz4(2 * np.pi * i / n1, 0.7) for i in range(n1)])
    frames, _ = wo.occupied_frames(Hl, 2)
    W = wo.wilson_matrix(frames)
    m = 2
    acc = [[1.0 + 0j if a == b else 0j for b in range(m)] for a in range(m)]
    detsum = 0.0
    for j in range(n1):
        A, B = frames[j], frames[(j + 1) % n1]
        M = [[sum(np.conj(A[r, a]) * B[r, b] for r in range(4)) for b in range(m)] for a in range(m)]
        detsum += np.angle(M[0][0] * M[1][1] - M[0][1] * M[1][0])
        acc = [[sum(acc[a][c] * M[c][b] for c in range(m)) for b in range(m)] for a in range(m)]
    assert np.allclose(np.array(acc), W, atol=1e-13)
    th, _ = wo.eigenphases(W)
    assert abs(wo.wrap_pi(np.sum(th) - detsum)) < 1e-11
    # 2x2 closed form: lambda = tr/2 +- sqrt(tr^2/4 - det)
    tr, det = W[0, 0] + W[1, 1], W[0, 0] * W[1, 1] - W[0, 1] * W[1, 0]
    lam = np.array([tr / 2 + np.sqrt(tr * tr / 4 - det), tr / 2 - np.sqrt(tr * tr / 4 - det)])
    assert wo.circ_sorted_distance(th, np.angle(lam)) < 1e-10


def test_path_ordering_matters_and_direction_conjugates():
    """Reversing the path conjugates the spectrum of W (W -> W^dagger up to similarity); a
    scrambled order does not give the same phases (non-Abelian)."""
    parts = wl.config5_parts(norb_spatial=4, delta=3.0)
    n1 = 12
    Hl = np.array([wl.assemble_config5(parts, 2 * np.pi * np.array([0.13, 0.41, l / n1]))
                   for l in range(n1)])
    frames, mg = wo.occupied_frames(Hl, 4)
    assert mg > 0.2
    th, _ = wo.eigenphases(wo.wilson_matrix(frames))
    rev = [frames[0]] + frames[:0:-1]
    thr, _ = wo.eigenphases(wo.wilson_matrix(rev))
    assert wo.circ_sorted_distance(th, -thr) < 1e-10
    perm = [frames[i] for i in (0, 2, 1, 3, 5, 4, 6, 7, 9, 8, 10, 11)]
    thp, _ = wo.eigenphases(wo.wilson_matrix(perm))
    assert wo.circ_sorted_distance(th, thp) > 1e-4


# ------------------------------------------------------------------ gauge invariance, |lambda| -> 1
def _random_unitary(rng, m):
    Z = rng.standard_normal((m, m)) + 1j * rng.standard_normal((m, m))
    Q, R = np.linalg.qr(Z)
    return Q * (np.diag(R) / np.abs(np.diag(R)))


def test_gauge_invariance_random_unitary_per_k():
    rng = np.random.default_rng(7)
    parts = wl.config5_parts(norb_spatial=8, delta=3.0)
    n1 = 15
    Hl = np.array([wl.assemble_config5(parts, 2 * np.pi * np.array([0.3, 0.8, l / n1]))
                   for l in range(n1)])
    frames, _ = wo.occupied_frames(Hl, 8)
    th, ab = wo.eigenphases(wo.wilson_matrix(frames))
    scr = [U @ _random_unitary(rng, 8) for U in frames]
    th2, ab2 = wo.eigenphases(wo.wilson_matrix(scr))
    assert wo.circ_sorted_distance(th, th2) < 1e-12
    assert np.allclose(np.sort(ab), np.sort(ab2), atol=1e-12)


def test_eigenvalue_modulus_tends_to_one_on_dense_grids():
    dev = []
    for n1 in (25, 100, 400):
        Hl = np.array([wl.bhz4(2 * np.pi * i / n1, 1.1) for i in range(n1)])
        _, ab, _ = wo.wilson_loop(Hl, 2)
        assert np.all(ab <= 1 + 1e-12)
        dev.append(1 - ab.min())
    assert dev[0] > dev[1] > dev[2]
    assert dev[2] < 0.02 and dev[1] / dev[2] > 3.0  # 1 - |lambda| = O(1/N1)


# ------------------------------------------------------------------ eigenvalues (S1)
def test_eigenvalues_closed_forms():
    rng = np.random.default_rng(3)
    for _ in range(5):
        kx, ky = rng.uniform(0, 2 * np.pi, 2)
        E, _ = wo.eigh_batched(wl.bhz4(kx, ky)[None])
        e = np.sqrt(np.sin(kx) ** 2 + np.sin(ky) ** 2 + (1 - np.cos(kx) - np.cos(ky)) ** 2)
        assert np.allclose(E[0], [-e, -e, e, e], atol=1e-13)
        E, _ = wo.eigh_batched(wl.bbh(kx, ky, 0.5, 1.0)[None])
        e = np.sqrt((0.5 + np.cos(kx)) ** 2 + np.sin(kx) ** 2 + (0.5 + np.cos(ky)) ** 2 + np.sin(ky) ** 2)
        assert np.allclose(E[0], [-e, -e, e, e], atol=1e-13)


def test_supercell_spectrum_is_folded_primitive_spectrum():
    """Clean L x L supercell at twist (t1,t2): spectrum = union over n of the 4-band spectra at
    k = 2 pi (t + n)/L (k = 2 pi n_x / L + theta_x / L)."""
    L = 4
    parts = wl.bhz_supercell_parts(L)
    t1, t2 = 0.23, 0.61
    E, U = wo.eigh_batched(wl.assemble_supercell(parts, t1, t2)[None])
    ref = []
    for nx in range(L):
        for ny in range(L):
            kx, ky = 2 * np.pi * (t1 + nx) / L, 2 * np.pi * (t2 + ny) / L
            e = np.sqrt(np.sin(kx) ** 2 + np.sin(ky) ** 2 + (1 - np.cos(kx) - np.cos(ky)) ** 2)
            ref += [-e, -e, e, e]
    assert np.allclose(E[0], np.sort(ref), atol=1e-12)
    H = wl.assemble_supercell(parts, t1, t2)
    assert np.allclose(H, H.conj().T)
    assert abs(np.trace(H).real - E[0].sum()) < 1e-10
    assert np.linalg.norm(H @ U[0] - U[0] * E[0]) < 1e-12
    # periodic gauge: H(t + 1) = H(t)
    assert np.allclose(wl.assemble_supercell(parts, t1 + 1, t2), H)


def test_zheev_agrees_with_zheevd_R14():
    import scipy.linalg as sl
    H = wl.assemble_supercell(wl.config3_parts(0, L=5), 0.3, 0.7)
    E, _ = wo.eigh_batched(H[None])
    Eev = sl.eigh(H, eigvals_only=True, driver="ev")
    assert np.max(np.abs(E[0] - Eev)) < 1e-13 * np.linalg.norm(H, 2) * 10


# ------------------------------------------------------------------ folding identity (large-m product)
def test_supercell_folding_identity():
    """Exact at finite N1.  Clean L x 1... here L x L supercell in the *position* gauge along x
    with closing Phi = e^{-i 2 pi x / L}: {lambda^L} = eigenvalues of the primitive 4-band loop
    with L N1 points at ky = 2 pi (t2 + n)/L, each repeated L times."""
    L, n1 = 3, 7
    parts = wl.bhz_supercell_parts(L)
    t2 = 0.37
    xs = np.repeat(np.arange(L), L * 4).astype(float)  # x coordinate of each orbital (site = L x + y)
    lam_super = []
    frames = []
    for i in range(n1):
        t1 = i / n1
        Hper = wl.assemble_supercell(parts, t1, t2)
        D = np.exp(1j * 2 * np.pi * t1 * xs / L)  # position gauge: H_pos = D^dagger H D
        Hpos = (np.conj(D)[:, None] * Hper) * D[None, :]
        E, V = np.linalg.eigh(Hpos)
        frames.append(V[:, : 2 * L * L])
    phi = np.exp(-1j * 2 * np.pi * xs / L)
    W = wo.wilson_matrix(frames, close=phi)
    lam_super = np.linalg.eigvals(W) ** L
    lam_prim = []
    for ny in range(L):
        ky = 2 * np.pi * (t2 + ny) / L
        Hl = np.array([wl.bhz4(2 * np.pi * i / (L * n1), ky) for i in range(L * n1)])
        fr, _ = wo.occupied_frames(Hl, 2)
        lam_prim += list(np.linalg.eigvals(wo.wilson_matrix(fr))) * L
    lam_prim = np.array(lam_prim)
    # optimal matching of two multisets of complex numbers
    from scipy.optimize import linear_sum_assignment
    cost = np.abs(lam_super[:, None] - lam_prim[None, :])
    r, c = linear_sum_assignment(cost)
    assert cost[r, c].max() < 1e-11


# ------------------------------------------------------------------ spin-resolved (S6)
def test_bhz_spin_resolved_windings_and_block_reduction():
    n1, n2 = 60, 41
    H = wl.config1_grid(n1, n2)
    S = wl.bhz4_spin_z()
    lo, hi, pso = wo.spin_resolved_surface(H[None], 2, 1, S)
    assert np.allclose(np.abs(pso), GOLD["pso_abs_eigenvalue_no_soc"], atol=1e-12)  # [H,S]=0
    w_lo, w_hi = wo.winding(lo), wo.winding(hi)
    assert abs(abs(w_lo) - GOLD["bhz_sector_abs_winding"]) < 1e-10
    assert abs(w_lo + w_hi - GOLD["bhz_total_winding"]) < 1e-10
    th, _, _ = wo.wilson_surface(H[None], 2, 1)
    assert abs(wo.winding(th) - GOLD["bhz_total_winding"]) < 1e-10
    # R11: lower sector (S_z = -1) winds +1 => C_down = -1, C_up = +1, C_s = +1 (paper sign)
    assert round(w_lo) == 1 and round(w_hi) == -1
    # band window [2, 4) (NEXT-3): within each spin block the two bands carry opposite Chern numbers,
    # so the unoccupied pair winds the other way, sector by sector
    ulo, uhi, upso = wo.spin_resolved_surface(H[None], 4, 1, S, band_lo=2)
    assert np.allclose(np.abs(upso), GOLD["pso_abs_eigenvalue_no_soc"], atol=1e-12)
    assert round(wo.winding(ulo)) == -1 and round(wo.winding(uhi)) == 1
    # block reduction: spin-down block (indices 1,3) is -sin kx sx + sin ky sy + M sz etc.
    for j in (0, 5, 17):
        ky = 2 * np.pi * j / n2
        for sgn, sector in ((-1.0, lo), (+1.0, hi)):
            Hl = np.array([sgn * np.sin(2 * np.pi * i / n1) * wl.sx + np.sin(ky) * wl.sy
                           + (1 - np.cos(2 * np.pi * i / n1) - np.cos(ky)) * wl.sz for i in range(n1)])
            tb, _, _ = wo.wilson_loop(Hl, 1)
            assert abs(wo.wrap_pi(tb[0] - sector[j, 0])) < 1e-10
    # the union of the sector phases is the full spectrum when [H,S]=0
    for j in range(n2):
        assert wo.circ_sorted_distance(th[j], np.concatenate([lo[j], hi[j]])) < 1e-10


def test_spin_resolved_with_spin_mixing_keeps_quantized_sector_windings():
    """with spin-orbit coupling PSO eigenvalues leave +-1 but stay gapped."""
    n1, n2 = 40, 31
    H = wl.config1_grid(n1, n2)
    mix = 0.3 * np.kron(wl.sy, wl.sx)  # anticommutes with neither mass term entirely; breaks S_z
    H = H + mix
    S = wl.bhz4_spin_z()
    lo, hi, pso = wo.spin_resolved_surface(H[None], 2, 1, S)
    assert np.abs(pso).min() < 1 - 1e-2 and np.abs(pso).min() > 0.2  # left +-1, still gapped
    assert abs(abs(wo.winding(lo)) - 1) < 1e-9 and abs(wo.winding(lo) + wo.winding(hi)) < 1e-9


# ------------------------------------------------------------------ nested (S5)
@pytest.mark.parametrize("gamma,key", [(0.5, "bbh_nested_polarization_topological"),
                                       (1.5, "bbh_nested_polarization_trivial")])
def test_bbh_nested_polarization(gamma, key):
    n = 40
    H = wl.config2_grid(n, n, gamma=gamma)
    for base in (0, 11):
        for band in (0, 1):
            th1, thn = wo.nested_wilson(H, 2, base=base, wb_lo=band, wb_hi=band + 1)
            assert wo.nested_polarization(thn) == GOLD[key]
            p = (-thn[0] / (2 * np.pi)) % 1.0
            assert min(abs(p - GOLD[key]), abs(p - GOLD[key] - 1), abs(p - GOLD[key] + 1)) < 1e-9
    # Wannier bands are gapped at 0 and 1/2 and symmetric about 0
    nu = th1 / (2 * np.pi)
    assert np.all(np.abs(nu) > 0.02) and np.all(np.abs(nu) < 0.48)
    assert np.allclose(nu[:, 0], -nu[:, 1], atol=1e-10)


def test_chiral_hoti_eq9_validation_model():
    """NEXT-4, Eq. 9: (a) Delta_0 = 1, k_z = 0: the WCC spectrum is gapped (PAPER.md:142,
    Fig. 4(a)) although (b) |C_s| = 1 with s = sigma_3 x tau_3 = diag(1,-1,-1,1) and a PSO whose
    eigenvalues left +-1 but stay gapped; (c) Delta_0 = 0, k_z = 0 is the BHZ-like QSH
    plane with a gapless (connected) WCC spectrum; (d) the nested Wilson loop along k_y of
    the lower Wannier band is gapless as a function of k_z: it winds once (Fig. 4(b))."""
    n = 32
    S = wl.chiral_hoti_spin()
    assert np.array_equal(S, np.array([1.0, -1.0, -1.0, 1.0]))            # op = np.diag([1,-1,-1,1])
    H = wl.chiral_hoti_grid(n, n, [0.0], 1.0)
    th, _, mg = wo.wilson_surface(H, 2, 1)
    assert mg.min() > 1.0
    assert np.abs(th).min() > 0.3 and np.abs(th).max() < np.pi - 0.3        # (a) gaps around 0 and pi for all k_y
    assert wo.chern_number(th) == 0
    lo, hi, pso = wo.spin_resolved_surface(H, 2, 1, S)
    assert abs(wo.chern_number(lo)) == abs(wo.chern_number(hi)) == int(GOLD["hoti_abs_spin_chern"])   # (b)
    assert wo.chern_number(lo) + wo.chern_number(hi) == 0
    assert np.abs(np.abs(pso) - 1).max() > 1e-3 and (pso[..., 1] - pso[..., 0]).min() > 0.4
    H0 = wl.chiral_hoti_grid(n, 96, [0.0], 0.0)
    th0, _, _ = wo.wilson_surface(H0, 2, 1)
    pts = np.sort(np.mod(th0.ravel(), 2 * np.pi))
    assert np.diff(np.concatenate([pts, [pts[0] + 2 * np.pi]])).max() < 0.5   # (c) no empty arc: connected spectrum
    kzs = [j / 20 for j in range(20)]
    Hz = wl.chiral_hoti_grid(24, 24, kzs, 1.0)
    nested = np.array([wo.nested_wilson(Hz[a], 2)[1] for a in range(20)])   # [20][1]
    assert abs(wo.chern_number(nested)) == int(GOLD["hoti_nested_abs_winding"])   # (d)


def test_nested_closing_phases_chiral_position_gauge():
    """close1 / close2 of nested_wilson.  BBH is chiral (tau_3 x sigma_0
    anticommutes with H), so every vector of the occupied space has weight exactly 1/2 on the orbitals
    {0, 1} and 1/2 on {2, 3}.  Putting those two pairs at the positions a and b along an axis therefore shifts
    every Berry phase along that axis by exactly -2 pi (a + b) / 2 when the embedding phase
    Phi = exp(-2 pi i r) closes the loop -- at any grid size -- as in the SSH pin above.  Dropping Phi_2
    gives back p = 1/2, conj(Phi_2) gives 0.9: both are caught."""
    n = 24
    H = wl.config2_grid(n, n, gamma=0.5)
    th1_per, thn_per = wo.nested_wilson(H, 2)
    r = np.array([0.3, 0.3, -0.1, -0.1])   # (a + b) / 2 = 0.1
    zero = np.zeros(4)
    # position gauge along k2 only: first-level phases untouched, nested polarization 1/2 + 0.1
    Hy, _, c2 = wl.position_gauge_plane(H, zero, r)
    for band in (0, 1):
        th1, thn = wo.nested_wilson(Hy, 2, wb_lo=band, wb_hi=band + 1, close2=c2)
        assert abs(((-thn[0] / (2 * np.pi)) % 1.0) - (GOLD["bbh_nested_polarization_topological"] + 0.1)) < 1e-10
        assert max(wo.circ_sorted_distance(th1[j], th1_per[j]) for j in range(n)) < 1e-11
    # position gauge along k1 only: det W (the sum of the first-level phases, two occupied vectors) moves by
    # -2 pi 2 (a + b) / 2 exactly, the nested polarization stays 1/2
    Hx, c1, _ = wl.position_gauge_plane(H, r, zero)
    th1, thn = wo.nested_wilson(Hx, 2, close1=c1)
    assert np.abs(wo.wrap_pi(th1.sum(axis=1) - th1_per.sum(axis=1) + 2 * np.pi * 0.2)).max() < 1e-11
    assert abs(((-thn[0] / (2 * np.pi)) % 1.0) - GOLD["bbh_nested_polarization_topological"]) < 1e-10
    # both axes
    Hxy, c1, c2 = wl.position_gauge_plane(H, r, 0.5 * r)
    th1, thn = wo.nested_wilson(Hxy, 2, close1=c1, close2=c2)
    assert abs(((-thn[0] / (2 * np.pi)) % 1.0) - (GOLD["bbh_nested_polarization_topological"] + 0.05)) < 1e-10
    # a missing Phi_1 is caught at both levels
    th1_no, thn_no = wo.nested_wilson(Hx, 2)
    assert np.abs(wo.wrap_pi(th1_no.sum(axis=1) - th1_per.sum(axis=1) + 2 * np.pi * 0.2)).max() > 0.1
    assert abs(((-thn_no[0] / (2 * np.pi)) % 1.0) - GOLD["bbh_nested_polarization_topological"]) > 1e-2


def test_nested_base_point_rephasing_exact_identity():
    """The ``base > 0`` branch of nested_wilson with a closing phase (R6, R9): a loop that starts at grid
    index b wraps past the zone boundary, and the wrapped frames carry Phi_1.  Exact identity: with
    D(k) = exp(i k r), H_pos(k_{i+b}) = C^dagger [D^dagger(k_i) H_per(k_{i+b}) D(k_i)] C, C = D(k_b)
    constant, so the base-b loop of H_pos equals the base-0 loop of the position-gauge version of the
    ROLLED periodic grid, first-level phases and nested phases alike (asymmetric positions, generic bands)."""
    n, b = 14, 5
    H = wl.config2_grid(n, n, gamma=0.7)
    r1 = np.array([0.11, 0.37, -0.23, 0.41])
    r2 = np.array([0.29, -0.13, 0.07, 0.33])
    Hp, c1, c2 = wl.position_gauge_plane(H, r1, r2)
    Hrolled, _, _ = wl.position_gauge_plane(H, r1, r2, shift1=b)
    for band in (0, 1):
        ta, na = wo.nested_wilson(Hp, 2, base=b, wb_lo=band, wb_hi=band + 1, close1=c1, close2=c2)
        tb, nb = wo.nested_wilson(Hrolled, 2, base=0, wb_lo=band, wb_hi=band + 1, close1=c1, close2=c2)
        assert max(wo.circ_sorted_distance(ta[j], tb[j]) for j in range(n)) < 1e-11
        assert abs(wo.wrap_pi(na[0] - nb[0])) < 1e-10
    # the identity is sharp: without the closing phase the base-b loop is a different object
    tc, nc = wo.nested_wilson(Hp, 2, base=b, close2=c2)
    assert max(wo.circ_sorted_distance(tc[j], tb[j]) for j in range(n)) > 1e-3


def test_nested_theta_cut_relabels_the_wannier_bands():
    """R9: Wannier bands are numbered by ascending phase on the branch (theta_cut - 2 pi, theta_cut].  The
    two Wannier bands of the chiral HOTI slice (Eq. 9) sit at +-nu with 0 < nu < 1/2: with
    the cut at pi band 0 is -nu, with the cut at 0 (branch (-2 pi, 0]) band 0 is +nu, and their nested
    phases at generic k_z are +-theta, not equal -- so the cut is observable."""
    Hz = wl.chiral_hoti_grid(16, 16, [0.1], 1.0)[0]
    th1, n_pi_0 = wo.nested_wilson(Hz, 2, wb_lo=0, wb_hi=1, theta_cut=np.pi)
    _, n_pi_1 = wo.nested_wilson(Hz, 2, wb_lo=1, wb_hi=2, theta_cut=np.pi)
    _, n_0_0 = wo.nested_wilson(Hz, 2, wb_lo=0, wb_hi=1, theta_cut=0.0)
    _, n_0_1 = wo.nested_wilson(Hz, 2, wb_lo=1, wb_hi=2, theta_cut=0.0)
    assert np.all(th1[:, 0] < -0.05) and np.all(th1[:, 1] > 0.05)        # the premise: bands at -nu and +nu
    assert abs(wo.wrap_pi(n_pi_0[0] - n_pi_1[0])) > 0.1                   # the two bands differ ...
    assert abs(wo.wrap_pi(n_0_0[0] - n_pi_1[0])) < 1e-10                  # ... and the cut swaps their numbers
    assert abs(wo.wrap_pi(n_0_1[0] - n_pi_0[0])) < 1e-10
    # both bands together: the selected span is the whole occupied space for either cut
    _, n_both_pi = wo.nested_wilson(Hz, 2, wb_lo=0, wb_hi=2, theta_cut=np.pi)
    _, n_both_0 = wo.nested_wilson(Hz, 2, wb_lo=0, wb_hi=2, theta_cut=0.0)
    assert wo.circ_sorted_distance(n_both_pi, n_both_0) < 1e-10


def test_spin_resolved_uneven_split_and_dense_spin_operator():
    """m_lo != m / 2 (R10) and the dense-S branch of projected_spin.  BHZ plus one
    decoupled occupied spin-down orbital, n_occ = 3: the PSO spectrum is (-1, -1, +1), so the sectors have
    the sizes 2 and 1.  Block reduction: the lower sector's phases are the union of the spin-down BHZ block's
    loop and the Abelian loop of the extra orbital (a k-independent vector: phase 0), the upper sector is
    the spin-up block; sector windings -+1.  The same model in a randomly rotated basis has
    a dense Hermitian S and must give the same phases."""
    n1, n2 = 40, 21
    H = wl.bhz4_plus_band_grid(n1, n2)
    S = wl.bhz4_plus_band_spin_z()
    lo, hi, pso = wo.spin_resolved_surface(H[None], 3, 1, S, m_lo=2)
    assert lo.shape == (n2, 2) and hi.shape == (n2, 1)
    assert np.abs(pso[..., :2] + GOLD["pso_abs_eigenvalue_no_soc"]).max() < 1e-12 and np.abs(pso[..., 2] - 1).max() < 1e-12
    up = [0, 2]; dn = [1, 3]
    th_up, _, _ = wo.wilson_surface(H[None][..., up, :][..., :, up], 1, 1)
    th_dn, _, _ = wo.wilson_surface(H[None][..., dn, :][..., :, dn], 1, 1)
    for j in range(n2):
        assert wo.circ_sorted_distance(hi[j], th_up[j]) < 1e-10
        assert wo.circ_sorted_distance(lo[j], np.sort(np.array([th_dn[j, 0], 0.0]))) < 1e-10
    assert abs(abs(wo.winding(lo)) - GOLD["bhz_sector_abs_winding"]) < 1e-9
    assert abs(wo.winding(lo) + wo.winding(hi)) < 1e-9
    # default split (m_lo = 1) cuts the degenerate pair of -1 eigenvalues: a different, ill-defined object
    Hr, Sr = wl.rotated_basis(H, S)
    assert np.abs(Sr - np.diag(np.diag(Sr))).max() > 0.1                     # S really is dense
    lo_r, hi_r, pso_r = wo.spin_resolved_surface(Hr[None], 3, 1, Sr, m_lo=2)
    assert np.abs(pso_r - pso).max() < 1e-11
    for j in range(n2):
        assert wo.circ_sorted_distance(lo_r[j], lo[j]) < 1e-10 and wo.circ_sorted_distance(hi_r[j], hi[j]) < 1e-10
    # a transposed or conjugated S is a different operator in the rotated basis and breaks the +-1 spectrum
    _, _, pso_t = wo.spin_resolved_surface(Hr[None][:, :2], 3, 1, Sr.T, m_lo=2)
    assert np.abs(np.abs(pso_t) - 1).max() > 1e-3


def test_nested_first_level_matches_plain_surface():
    H = wl.config2_grid(24, 20)
    th1, _ = wo.nested_wilson(H, 2)
    th, _, _ = wo.wilson_surface(H[None], 2, 1)
    for j in range(20):
        assert wo.circ_sorted_distance(th1[j], th[j]) < 1e-12


# ------------------------------------------------------------------ comparator and invariants
def test_comparator_handles_cut_and_degenerate_clusters():
    a = np.array([-np.pi + 1e-12, 0.0, 0.0, 0.0, 1.0])
    b = np.array([0.0, 0.0, 0.0, 1.0, np.pi - 1e-12])
    assert wo.circ_sorted_distance(a, b) < 1e-11
    assert abs(wo.circ_sorted_distance(np.array([0.1, 0.5]), np.array([0.1, 0.6])) - 0.1) < 1e-15


def test_winding_counts_turns():
    i = np.arange(50)
    for w in (-2, -1, 0, 1, 3):
        th = wo.wrap_pi(2 * np.pi * w * i / 50 + 0.3)[:, None]
        assert abs(wo.winding(th) - w) < 1e-12


# ------------------------------------------------------------------ workload sanity (harness asserts)
def test_config5_gap_and_hermiticity():
    parts = wl.config5_parts()
    rng = np.random.default_rng(0)
    gaps = []
    for _ in range(40):
        k = rng.uniform(0, 2 * np.pi, 3)
        H = wl.assemble_config5(parts, k)
        assert np.allclose(H, H.conj().T)
        E = np.linalg.eigvalsh(H)
        gaps.append(E[32] - E[31])
    assert min(gaps) >= 0.2


def test_config3_and_4_structure():
    p3 = wl.config3_parts(0, L=4)
    H = wl.assemble_supercell(p3, 0.1, 0.2)
    assert np.allclose(H, H.conj().T)
    on = wl.config4_onsite(20)
    nz = [(x, y) for x in range(20) for y in range(20) if np.abs(on[x, y]).max() > 0]
    assert len(nz) == 20
    for x, y in nz:
        assert np.allclose(np.abs(np.diag(on[x, y])), 0.3)
    S = wl.supercell_spin_z(3)
    assert S.shape == (36,) and set(S) == {1.0, -1.0}
