"""Batched sign-iteration microbench of BASELINE.json configs[4] (the analogue of the paper's Fig. 6,
PAPER.md:268): uniform batches of random symmetric gapped matrices A = Q diag(lam) Q^T, n in
{256, 512, 1024, 2048, 4096}, batch such that one batched product is ~2^34 FLOP (times --scale),
X0 = A / max|lam|, residual stop rule (reading 9).  Prints one line per (n, precision):
iterations, kernel time of the sign-iteration launch (CUDA events inside libnolsm) and TFLOP/s on
2 n^3 per executed product, plus max |X - sign(A)| against the construction.

    python -m paper_2104_08245_b200.microbench [--scale 16] [--sizes 256,512,1024] [--flags 0]

To keep the host-side QR short, a batch holds at most --distinct different matrices, repeated.
"""
import argparse
import json
import sys

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--sizes", default="256,512,1024,2048,4096")
    ap.add_argument("--scale", type=int, default=1, help="batch = scale * 2^34 / (2 n^3) (at least 1)")
    ap.add_argument("--distinct", type=int, default=4)
    ap.add_argument("--flags", type=int, default=0)
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--group", type=int, default=0, help="nolsm_config.group: window of submatrices in flight (0: default)")
    ap.add_argument("--precisions", default="0,1", help="0 = FP16/FP32, 1 = FP32 quality")
    args = ap.parse_args()
    import torch
    import nolsm_inputs as gi
    from . import Context, Config, load_library
    load_library()
    if not torch.cuda.is_available():
        raise SystemExit("the microbench needs a CUDA device; there is no CPU fallback")
    for n in [int(x) for x in args.sizes.split(",")]:
        batch = max(1, args.scale * gi.microbench_batch(n))
        mats = [gi.make_gapped_symmetric(n, seed=5, index=i) for i in range(min(batch, args.distinct))]
        idx = np.arange(batch) % len(mats)
        a = torch.as_tensor(np.stack([m[0] for m in mats]))[torch.as_tensor(idx)].contiguous().cuda()
        scale = torch.as_tensor(np.array([np.abs(mats[i][2]).max() for i in idx], dtype=np.float32)).cuda()
        signs = [(m[1] * np.sign(m[2])[None, :]) @ m[1].T for m in mats]
        for precision in [int(x) for x in args.precisions.split(",")]:
            ctx = Context(Config(precision=precision, flags=args.flags, group=args.group))
            best, stats, x = None, None, None
            for _ in range(args.reps):
                x, st = ctx.sign_dense_batched(a, scale)
                if best is None or st.ms_chain < best:
                    best, stats = st.ms_chain, st
            err = max(float(np.abs(x[i].cpu().numpy() - signs[idx[i]]).max()) for i in range(min(batch, len(mats))))
            print(json.dumps({"n": n, "batch": batch, "precision": "fp16/fp32" if precision == 0 else "fp32 (split fp16)",
                              "iterations": [stats.iter_min, stats.iter_max], "unconverged": stats.n_unconverged,
                              "ms_kernel": round(best, 4), "sm_ghz": round(stats.chain_mcycles / max(best, 1e-9), 3), "tflops": round(stats.flops_sign / best * 1e-9, 1),
                              "max_abs_err_vs_construction": err, "engine_flags": args.flags, "group": args.group}), flush=True)
            ctx.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
