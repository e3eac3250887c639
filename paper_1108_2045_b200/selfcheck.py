"""Self-check of an installation: a few small solves through the C ABI on cuda:0, every kernel family once.

    python -m paper_1108_2045_b200.selfcheck [--tiny]

Runs the five workloads' recipes at small sizes with the TMA-tiled kernels forced onto every level
(tiled_min_nodes=1: K_res, K_visit in 2-D and 3-D, the vectorised level changes, K_coarse), in plain-launch and
graph mode, the classic V cycle, the paper-literal mode, the mixed-precision loop and homg_solve, and checks that
every solve contracts its residual.  It is the command the compute-sanitizer records under profiles/ were taken
with (memcheck, racecheck, initcheck).  No oracle here: parity is tests/ (-m gpu).
"""
import sys

import numpy as np

from . import homg, inputs as I


def run(name, n, ncyc, **kw):
    cfg = I.CONFIGS[name] if I.CONFIGS[name].dims[0] == n else I.scaled(I.CONFIGS[name], n)
    inp = I.make_inputs(cfg)
    mixed = kw.get("mixed", False)
    if mixed:
        inp = {k: (None if v is None else v.astype(np.float64)) for k, v in inp.items()}
    s = homg.Solver(cfg.dims, cfg.levels, cfg.stencil, "f64" if mixed else cfg.dtype, omega=cfg.omega,
                    max_iters=cfg.max_iters, **kw)
    if inp["k"] is not None:
        s.set_coefficient(inp["k"])
    s.set_rhs(inp["f"])
    s.set_initial_guess(inp["u0"])
    if kw.get("vcycle") is None and not kw.get("literal") and not mixed:
        done, rel = s.solve(1e-30, ncyc)                      # the device-side loop, capped by max_cycles
        assert done == ncyc
    s.cycle(ncyc)
    hist = s.residual_history()
    final, rel = s.residual_norm()
    u = s.get_solution()
    s.destroy()
    assert np.isfinite(u).all() and np.isfinite(final)
    first = hist[1] if len(hist) > 1 else hist[0]             # (the first factor may exceed 1 from u0 = 0: DESIGN.md R15)
    assert final < first, (name, n, kw, hist, final)
    return final / hist[0]


def main(tiny=False):
    import torch
    assert torch.cuda.is_available(), "selfcheck needs a CUDA device (there is no CPU fallback)"
    n3, n2 = (17, 65) if tiny else (33, 257)
    out = []
    for name, n in (("cfg1", 129 if not tiny else 65), ("cfg2", n3), ("cfg3", n2), ("cfg4", n3), ("cfg5", n3)):
        out.append((name, n, "tiled", run(name, n, 3, tiled_min_nodes=1)))
        out.append((name, n, "default", run(name, n, 3)))
    out.append(("cfg2", n3, "no graph", run("cfg2", n3, 3, tiled_min_nodes=1, use_graph=0)))
    out.append(("cfg4", n3, "V(2,1)", run("cfg4", n3, 3, tiled_min_nodes=1, vcycle=(2, 1))))
    out.append(("cfg2", 17, "literal", run("cfg2", 17, 2, literal=True)))
    out.append(("cfg5", n3, "mixed", run("cfg5", n3, 3, tiled_min_nodes=1, mixed=True)))
    for name, n, what, rel in out:
        print(f"selfcheck {name}@{n} [{what}]: relative residual {rel:.3e}")
    print("selfcheck: ok")


if __name__ == "__main__":
    main(tiny="--tiny" in sys.argv)
