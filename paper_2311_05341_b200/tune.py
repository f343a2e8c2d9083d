"""A/B of the compiled kernel shapes on one GPU (the source of profiles/r02_tuning.md).

    python -m paper_2311_05341_b200.tune --config headline_u4 [--variants 16 22 23 ...] [--panels 0 86 ...]

Builds libdd.so with -DDD_TUNING (build.py --tuning: the extra shapes of kVariants in
csrc/dd_kernels.cu and the DD_FORCE_VARIANT / DD_PANEL environment variables exist only in such a
build), runs dd_execute a few times per choice on the config's synthetic block and prints one JSON
line per choice with the main kernel's CUDA-event time (dd_plan_kernel_times).  Every choice must
reproduce the first one's output bit for bit (parity against the oracle is tests/'s job).
Rebuild the default library afterwards: python -m paper_2311_05341_b200.build --force
"""
from __future__ import annotations

import argparse
import json
import os


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="headline")
    ap.add_argument("--variants", type=int, nargs="*", default=[-1], help="kVariants indices (-1 = the automatic choice)")
    ap.add_argument("--panels", type=int, nargs="*", default=[0], help="DM blocks per rasterisation panel (0 = the plan's choice)")
    ap.add_argument("--reps", type=int, default=4)
    args = ap.parse_args()
    import torch
    from . import build
    build.build(tuning=True)
    from . import binding as B, workloads as W
    cfg = W.ALL_CONFIGS[args.config]
    torch.cuda.set_device(0)
    x = W.noise_torch(cfg, "cuda")
    odt = torch.float32 if cfg.in_dtype == W.F32 else torch.int32
    ref = None
    for v in args.variants:
        for pn in args.panels:
            os.environ.pop("DD_FORCE_VARIANT", None)
            os.environ.pop("DD_PANEL", None)
            if v >= 0:
                os.environ["DD_FORCE_VARIANT"] = str(v)
            if pn > 0:
                os.environ["DD_PANEL"] = str(pn)
            try:
                plan = B.Plan(cfg.nchans, cfg.nsamps, cfg.f_high, cfg.chan_bw, cfg.tsamp, cfg.dm_list, cfg.in_dtype)
            except B.DDError as e:
                print(json.dumps({"config": cfg.name, "variant": v, "panel": pn, "error": str(e)}), flush=True)
                continue
            out = torch.empty((plan.ndm, plan.out_len), dtype=odt, device="cuda")
            plan.set_timing(True)
            for _ in range(args.reps):
                plan.execute(x, out)
            torch.cuda.synchronize()
            _, mn = plan.kernel_times(max(1, args.reps - 1))
            if ref is None:
                ref = out.clone()
            adds = plan.ndm * plan.out_len * cfg.nchans
            print(json.dumps({"config": cfg.name, "variant": v, "panel": pn or plan.info("PANEL"),
                              "tile": "D_DM=%d D_J=%d CH=%d stages=%d smem=%d threads=%d" % (
                                  plan.info("D_DM"), plan.info("D_J"), plan.info("CH"), plan.info("NSTAGE"),
                                  plan.info("SMEM_BYTES"), plan.info("THREADS")),
                              "kernel_ms": round(float(mn.mean()), 4),
                              "T_adds_per_s": round(adds / (float(mn.mean()) * 1e-3) / 1e12, 3),
                              "same_output_as_first": bool(torch.equal(ref, out))}), flush=True)
            plan.destroy()
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
