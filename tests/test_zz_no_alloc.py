"""tddft_gram_static (include/tddft.h): the Gram matrix with its split-k partial sums in the library's file-scope device array
instead of the context's arena, for callers that cannot call cudaMalloc.  Checked against the existing path (tddft_gram) on
calls in a row that share the array.  Collected last on purpose (file name): a failure here must not hide the parity tests."""
import numpy as np
import pytest

from helpers import Case

pytestmark = pytest.mark.gpu

TRI = [[7.0, 0, 0], [0.9, 7.4, 0], [0.5, -0.4, 6.6]]
TOL = 1e-12      # tolerance of test_gram_matches_oracle, relative to the largest entry


def _vectors(case, m, nblk):
    v = case.rng.standard_normal((m, nblk, case.npwh)) + 1j * case.rng.standard_normal((m, nblk, case.npwh))
    v[:, :, 0] = v[:, :, 0].real      # G = 0 of a real function
    return v.reshape(m, nblk * case.npwh)


def test_gram_static_matches_gram_on_calls_in_a_row():
    import torch
    from paper_2309_03513_b200 import binding as b
    case = Case(TRI, (12, 10, 9), 6.0, 2, (5, 4), 0.3, seed=911, oracle=False)
    ctx = case.ctx()
    nblk = -(-40000 // case.npwh)                 # K = 2 * n_complex > 80000 reals: ten or more k splits, so the scratch is in use
    n_complex = nblk * case.npwh
    assert 2 * n_complex // 8192 >= 9
    # 256 has its k splits cut down to the 4 MiB (8 < 2 * n_complex / 8192), the others keep those of tddft_gram; the small ones
    # run AFTER a large one, over its stale partial sums
    for call, m in enumerate((70, 5, 256, 22, 5)):
        V = torch.from_numpy(_vectors(case, m, nblk)).cuda()
        W = torch.from_numpy(_vectors(case, m, nblk)).cuda()
        ref = b.tddft_gram(ctx, V, W, m, n_complex)                      # existing path: arena scratch, host result
        G = torch.full((m, m), float("nan"), dtype=torch.float64, device="cuda")
        G2 = torch.full((m, m), float("nan"), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        b.tddft_gram_static(ctx, V, W, m, n_complex, G)
        # a second call on the same inputs, straight after: the array now holds this call's own partial sums
        b.tddft_gram_static(ctx, V, W, m, n_complex, G2)
        torch.cuda.synchronize()
        if call > 0:      # the very first call may load the module that holds the array
            assert torch.cuda.mem_get_info()[0] == free0, "tddft_gram_static took device memory"
        got = G.cpu().numpy()
        assert np.all(np.isfinite(got))
        assert np.max(np.abs(got - ref)) < TOL * np.max(np.abs(ref)), (call, m)
        if (2 * n_complex // 8192) * m * m <= (1 << 19):
            assert np.array_equal(got, ref), (call, m)                   # same splits, same kernels: same bits
        assert np.array_equal(G2.cpu().numpy(), got), (call, m)


def test_gram_static_rejects_sizes_beyond_the_scratch():
    import torch
    from paper_2309_03513_b200 import binding as b
    case = Case(TRI, (12, 10, 9), 6.0, 2, (5, 4), 0.3, seed=912, oracle=False)
    ctx = case.ctx()
    m = b.TDDFT_GRAM_STATIC_MAX_M + 1
    V = torch.zeros((m, case.npwh), dtype=torch.complex128, device="cuda")
    G = torch.zeros((m, m), dtype=torch.float64, device="cuda")
    with pytest.raises(b.TddftError) as e:
        b.tddft_gram_static(ctx, V, V, m, case.npwh, G)
    assert "256" in str(e.value) and "limit" in str(e.value)
    # the context is still usable
    m = 3
    V = torch.from_numpy(_vectors(case, m, 2)).cuda()
    G = torch.zeros((m, m), dtype=torch.float64, device="cuda")
    b.tddft_gram_static(ctx, V, V, m, 2 * case.npwh, G)
    torch.cuda.synchronize()
    assert np.allclose(G.cpu().numpy(), b.tddft_gram(ctx, V, V, m, 2 * case.npwh), rtol=0, atol=1e-12 * float(G.abs().max()))
