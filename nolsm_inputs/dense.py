"""Dense microbench inputs of BASELINE.json:configs[4]: random symmetric gapped matrices
A = Q diag(lam) Q^T with Q Haar-orthogonal, |lam| ~ U[0.05, 1], independent random signs.
Returns the factors too, so a checker knows the spectrum by construction.  Inputs only."""
import numpy as np

from . import rng as _rng


def make_gapped_symmetric(n, seed, index=0, lo=0.05, hi=1.0):
    """Returns (A float32 [n,n], Q float64 [n,n], lam float64 [n])."""
    ctr = np.arange(n * n, dtype=np.uint64)
    g = _rng.normal(seed, 1000 + 3 * index, ctr).reshape(n, n)
    q, r = np.linalg.qr(g)
    q = q * np.sign(np.diag(r))[None, :]
    k = np.arange(n, dtype=np.uint64)
    mag = lo + (hi - lo) * _rng.uniform_u53(seed, 1001 + 3 * index, k)
    sgn = np.where(_rng.uniform_u53(seed, 1002 + 3 * index, k) < 0.5, -1.0, 1.0)
    lam = mag * sgn
    a = (q * lam[None, :]) @ q.T
    a = 0.5 * (a + a.T)
    return a.astype(np.float32), q, lam


def microbench_batch(n, total_flops=2 ** 34):
    """Batch size so one batched GEMM is ~total_flops (reading of configs[4])."""
    return max(1, int(total_flops // (2 * n ** 3)))
