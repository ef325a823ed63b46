"""Launch one step of the cycle repeatedly on a synthetic workload (for ncu / timing).

    python -m paper_2605_30082_b200.profile_driver --step sweep2 --workload config4 --reps 3

steps: sweep4, sweep2, sweep1 (that many sweeps on --level), sweep_restrict (one sweep with the
residual + restriction tail), vcycle, residual, solve.  Prints the average
CUDA-event time per repetition.  Uses only the public binding and the workload generator.
"""
import argparse
import sys
from pathlib import Path

sys.path.insert(0, str(Path(__file__).resolve().parent.parent))


def main():
    import torch

    import paper_2605_30082_b200 as mgpkg
    from paper_2605_30082_b200 import binding as B
    from workloads import make_workload

    ap = argparse.ArgumentParser()
    ap.add_argument("--step", default="sweep2")
    ap.add_argument("--workload", default="config4")
    ap.add_argument("--level", type=int, default=0)
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--kernels", type=int, default=1)
    ap.add_argument("--graph", type=int, default=1)
    ap.add_argument("--fuse", type=int, default=2)
    args = ap.parse_args()
    body = args.workload[len("config"):]
    cfg, n = (body.split("@") + [None])[:2]
    w = make_workload(int(cfg), int(n) if n else None)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        g = mgpkg.Multigrid(w.n, w.h, w.bc, w.nu1, w.nu2, stream=st)
        g.set_option(B.MG_OPT_KERNELS, args.kernels)
        g.set_option(B.MG_OPT_GRAPH, args.graph)
        g.set_option(B.MG_OPT_SWEEP_FUSE, args.fuse)
        g.set_density(torch.from_numpy(w.rho).cuda())
        shp = g.level_shape(args.level)
        if args.level == 0:
            f = torch.from_numpy(w.rhs).cuda()
        else:
            f = torch.randn(shp, dtype=torch.float64, device="cuda")
        p = torch.zeros(shp, dtype=torch.float64, device="cuda")

        def run():
            if args.step == "sweep4":
                g.level_smooth(args.level, 4, f, p)
            elif args.step == "sweep2":
                g.level_smooth(args.level, 2, f, p)
            elif args.step == "sweep1":
                g.level_smooth(args.level, 1, f, p)
            elif args.step == "sweep_restrict":
                g.level_smooth_restrict(args.level, 1, f, p)
            elif args.step == "vcycle":
                g.vcycle(f, p)
            elif args.step == "residual":
                g.residual(f, p)
            elif args.step == "solve":
                p.zero_()
                g.solve(f, p, w.rtol, 60)
            else:
                raise SystemExit("unknown step")

        for _ in range(2):
            run()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for _ in range(args.reps):
            run()
        e1.record(st)
        torch.cuda.synchronize()
        print(f"{args.step} level {args.level} {w.name}: {e0.elapsed_time(e1) / args.reps:.4f} ms per rep")


if __name__ == "__main__":
    main()
