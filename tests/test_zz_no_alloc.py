"""be_eigh_batched_static (the entry point that allocates nothing: fixed static device scratch) against the
existing be_eigh_batched path on the same inputs, two calls in a row.

Collected last on purpose (file name): the suite runs with ``pytest -x``.  The test owns its context, so it passes
alone in a fresh process and after the other tests.  Both paths launch the same Jacobi kernel on the same data,
so the outputs are expected to agree to the bit; the assertion uses the eigenvalue tolerance of
tests/test_gpu_parity.py (1e-10 ||H||) and, for the eigenvectors, the residual / orthonormality bounds used there.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_2312_13051_b200 import workloads as wl

pytestmark = pytest.mark.gpu

E_TOL = 1e-10


def _random_hermitian(count, N, seed):
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((count, N, N)) + 1j * rng.standard_normal((count, N, N))
    return (A + A.conj().transpose(0, 2, 1)) / 2


def test_static_entry_matches_existing_path_twice():
    from paper_2312_13051_b200.binding import BerryEasyError, Context
    ctx = Context()
    try:
        # first call: config-1 slice (BHZ 4-band, 3 loops x 100 k-points, the two occupied vectors)
        H1 = np.ascontiguousarray(wl.config1_grid()[:3].reshape(-1, 4, 4))
        # second call, right after, other shape and MORE scratch than the first (stale contents must not matter)
        H2 = _random_hermitian(1777, 7, seed=20231213)
        for H, nv in ((H1, 2), (H2, 7), (H1, 2)):
            Hd = torch.from_numpy(H).cuda()
            count, N = H.shape[0], H.shape[1]
            E_ref, U_ref = ctx.eigh_batched(Hd, nv)
            E = torch.full((count, N), float("nan"), dtype=torch.float64, device="cuda")
            U = torch.full((count, N, nv), float("nan"), dtype=torch.complex128, device="cuda")
            info = torch.full((count,), -1, dtype=torch.int32, device="cuda")
            ctx.eigh_batched_static(Hd, E, U, info)
            torch.cuda.synchronize()
            assert int(info.abs().max()) == 0
            nrm = float(np.abs(np.linalg.eigvalsh(H)).max())
            assert float((E - E_ref).abs().max()) <= E_TOL * nrm
            assert float((U - U_ref).abs().max()) <= 1e-11 * N          # same kernel, same gauge
            Uh, Eh = U.cpu().numpy(), E.cpu().numpy()
            for c in range(0, count, max(count // 50, 1)):
                assert np.linalg.norm(H[c] @ Uh[c] - Uh[c] * Eh[c][:nv]) <= 1e-11 * nrm * N
                assert np.linalg.norm(Uh[c].conj().T @ Uh[c] - np.eye(nv)) <= 1e-11 * N
        # eigenvalues only: no scratch touched
        Hd = torch.from_numpy(H2).cuda()
        E_ref, _ = ctx.eigh_batched(Hd, 0)
        E = torch.empty((H2.shape[0], 7), dtype=torch.float64, device="cuda")
        ctx.eigh_batched_static(Hd, E)
        assert float((E - E_ref).abs().max()) <= E_TOL * float(np.abs(H2).sum(axis=2).max())
        # beyond the fixed scratch: a clear error, nothing enqueued
        big = (1 << 19) // 64 + 1
        Hb = torch.zeros((big, 8, 8), dtype=torch.complex128, device="cuda")
        Eb = torch.empty((big, 8), dtype=torch.float64, device="cuda")
        Ub = torch.empty((big, 8, 8), dtype=torch.complex128, device="cuda")
        with pytest.raises(BerryEasyError, match="static scratch"):
            ctx.eigh_batched_static(Hb, Eb, Ub)
        with pytest.raises(BerryEasyError):
            ctx.eigh_batched_static(torch.zeros((2, 9, 9), dtype=torch.complex128, device="cuda"),
                                    torch.empty((2, 9), dtype=torch.float64, device="cuda"))
    finally:
        ctx.close()
