"""GPU unit test of the per-atom linear-layer kernel: tcgen05 3xTF32 path vs an fp64 matmul (numpy) and vs the
plain fp32 SIMT path, on every (N, K) shape the F = 128 model uses, with ragged M and strided accumulate."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SHAPES = [(128, 128), (384, 128), (256, 128), (128, 256), (64, 128), (128, 64), (128, 384)]   # (N, K)


@pytest.mark.parametrize("M", [1, 127, 128, 129, 1000, 20000])
def test_gemm_tensor_core_matches_fp64(M):
    import torch
    import paper_2506_04055_b200 as P
    assert torch.cuda.is_available()
    rng = np.random.default_rng(M)
    for N, K in SHAPES:
        A = (rng.standard_normal((M, K)) * np.exp(rng.standard_normal((M, 1)))).astype(np.float32)
        W = (rng.standard_normal((N, K)) / np.sqrt(K)).astype(np.float32)
        b = rng.standard_normal(N).astype(np.float32)
        ref = A.astype(np.float64) @ W.astype(np.float64).T + b
        Ad = torch.from_numpy(A).cuda()
        C, used = P.debug_gemm(Ad, W, b, path=0)
        assert used, (M, N, K)
        C1, used1 = P.debug_gemm(Ad, W, b, path=1)
        assert not used1
        scale = np.abs(A).astype(np.float64) @ np.abs(W).astype(np.float64).T + np.abs(b)
        err_tc = np.abs(C.cpu().numpy() - ref) / scale
        err_simt = np.abs(C1.cpu().numpy() - ref) / scale
        assert err_simt.max() < 2e-6, (M, N, K, err_simt.max())
        assert err_tc.max() < 4e-6, (M, N, K, err_tc.max())          # 3xTF32: ~2^-21 per product
        # accumulate: C += A W^T
        C0 = torch.from_numpy(rng.standard_normal((M, N)).astype(np.float32)).cuda()
        ref2 = C0.cpu().numpy().astype(np.float64) + A.astype(np.float64) @ W.astype(np.float64).T
        C2, _ = P.debug_gemm(Ad, W, None, C_out=C0.clone(), accumulate=True, path=0)
        assert (np.abs(C2.cpu().numpy() - ref2) / (scale + np.abs(ref2))).max() < 4e-6


@pytest.mark.parametrize("M", [1, 127, 129, 1000, 20000])
def test_gemm_exact_slices_matches_fp64(M):
    """Forward path: integer-slice tensor-core kernel (exact accumulation).  Error is bounded relative to
    (row max of A) x (row max of W) x sqrt(K) x 2^-22; here checked against the same |A||W| scale as the fp32 kernel,
    and the mean signed error must show no truncation bias."""
    import torch
    import paper_2506_04055_b200 as P
    rng = np.random.default_rng(1000 + M)
    for N, K in [(128, 128), (384, 128), (256, 128), (128, 256), (64, 128)]:
        A = (rng.standard_normal((M, K)) * np.exp(rng.standard_normal((M, 1)))).astype(np.float32)
        if M > 2:
            A[1] = 0.0                                    # an all-zero row must give exactly the bias
        W = (rng.standard_normal((N, K)) / np.sqrt(K)).astype(np.float32)
        b = rng.standard_normal(N).astype(np.float32)
        ref = A.astype(np.float64) @ W.astype(np.float64).T + b
        Ad = torch.from_numpy(A).cuda()
        C, used = P.debug_gemm(Ad, W, b, path=2)
        assert used, (M, N, K)
        Ch = C.cpu().numpy()
        scale = np.abs(A).astype(np.float64) @ np.abs(W).astype(np.float64).T + np.abs(b)
        err = (Ch - ref) / scale
        assert np.abs(err).max() < 2e-6, (M, N, K, np.abs(err).max())
        if M > 2:
            assert np.array_equal(Ch[1], b)
        if M >= 1000:
            assert abs(err.mean()) < 2e-8, (M, N, K, err.mean())      # unbiased (3xTF32 chains sit near -1e-7)
        C0 = torch.from_numpy(rng.standard_normal((M, N)).astype(np.float32)).cuda()
        ref2 = C0.cpu().numpy().astype(np.float64) + A.astype(np.float64) @ W.astype(np.float64).T
        C2, _ = P.debug_gemm(Ad, W, None, C_out=C0.clone(), accumulate=True, path=2)
        assert (np.abs(C2.cpu().numpy() - ref2) / (scale + np.abs(ref2))).max() < 2e-6
