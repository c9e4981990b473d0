"""Launch every kernel of libdash_hash4d.so once on a tiny workload (for compute-sanitizer):
    compute-sanitizer --tool memcheck python tests/run_small_all_kernels.py
Not a pytest file; it checks nothing beyond finiteness — parity lives in tests/test_gpu_parity.py."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import numpy as np
import torch

import paper_2507_19141_b200 as dh
from dash_inputs import EncoderParams, make_queries_uniform


def main():
    rng = np.random.default_rng(0)
    for (L, F, T, dtype, n) in [(4, 2, 4096, "fp32", 1000), (5, 4, 5003, "fp16", 777), (3, 8, 1 << 12, "fp32", 130),
                                (6, 1, 1 << 13, "fp16", 257)]:
        enc = EncoderParams(L, F, T, 8, 200, 4, 40, dtype)
        xyz, t = make_queries_uniform(L, n)
        rows = rng.random((50, 3), dtype=np.float32)
        index = rng.integers(0, 50, n).astype(np.int32)
        table = rng.uniform(-1, 1, (L, T, F)).astype(np.float16 if dtype == "fp16" else np.float32)
        dout = rng.standard_normal((n, L * F)).astype(np.float32)
        d = lambda a: torch.from_numpy(a).cuda()
        for flags in (dh.FLAG_DENSE_COARSE, dh.FLAG_DENSE_COARSE | dh.FLAG_ZERO_GRAD,
                      dh.FLAG_DENSE_COARSE | dh.FLAG_DETERMINISTIC_BWD, dh.FLAG_VALIDATE_INPUTS):
            cfg = dh.config_from_params(enc, flags=flags)
            for (x, ix) in ((d(xyz), None), (d(rows), d(index))):
                out = dh.dash_hash4d_fwd(cfg, x, d(t), d(table), index=ix)
                dt = torch.empty((L, T, F), device="cuda")
                dh.dash_hash4d_zero(cfg, dt)
                dh.dash_hash4d_bwd(cfg, x, d(t), d(dout), dt, index=ix)
                dq = dh.dash_hash4d_bwd_input(cfg, x, d(t), d(table), d(dout), index=ix)
                idx, w = dh.dash_hash4d_indices(cfg, x, d(t), index=ix)
                torch.cuda.synchronize()
                assert torch.isfinite(out).all() and torch.isfinite(dt).all() and torch.isfinite(dq).all()
                assert int(idx.view(torch.int32).max()) < T
        # smoothness regulariser, G_3D, sparse Adam, render path (fused / two-pass / MLP alone), time slice
        cfg = dh.config_from_params(enc)
        x, tt, tab = d(xyz), d(t), d(table)
        eps = d((rng.random((n, 4), dtype=np.float32) - 0.5) * 1e-2)
        dt = torch.zeros((L, T, F), device="cuda")
        loss, _ = dh.dash_hash4d_smooth(cfg, x, tt, eps, tab, grad_scale=0.1, dtable=dt)
        o3 = dh.dash_hash3d_fwd(cfg, x, tab)
        dh.dash_hash3d_bwd(dh.with_flags(cfg, dh.FLAG_DENSE_COARSE | dh.FLAG_ZERO_GRAD), x, d(dout), dt)
        i3, _ = dh.dash_hash3d_indices(cfg, x)
        theta = tab.float().contiguous()
        m1, v1 = torch.zeros_like(theta), torch.zeros_like(theta)
        dh.dash_hash4d_adam_step(cfg, theta, dt, m1, v1, 1, table16=tab if dtype == "fp16" else None)
        widths = [L * F, 24, 10]
        mlp = dh.make_mlp_config(widths)
        prm = d(rng.uniform(-0.3, 0.3, dh.dash_mlp_param_count(mlp)).astype(np.float32))
        outs = []
        for fused in ("1", "0"):
            os.environ["DASH_DEFORM_FUSED"] = fused
            outs.append(dh.dash_deform_fwd(cfg, mlp, x, tt, tab, prm))
        os.environ.pop("DASH_DEFORM_FUSED")
        outs.append(dh.dash_mlp_fwd(mlp, dh.dash_hash4d_fwd(cfg, x, tt, tab), prm))
        if T & (T - 1) == 0:
            sl = dh.dash_hash4d_slice_t(cfg, tt[:1].contiguous(), tab)
            outs.append(dh.dash_hash4d_slice_fwd(cfg, x, sl))
            outs.append(dh.dash_deform_slice_fwd(cfg, mlp, x, sl, prm))
        torch.cuda.synchronize()
        for a in [loss, o3, theta, m1, v1] + outs:
            assert torch.isfinite(a).all()
        assert int(i3.max()) < T
    print("all kernels ran")


if __name__ == "__main__":
    main()
