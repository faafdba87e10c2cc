"""Runs a few steps of a named workload on cuda:0 and prints what happened -- a small driver for tools that wrap a whole
process (compute-sanitizer, ncu):

    python -m paper_2302_02474_b200.selfcheck C2 --steps 12 [--flags N]
"""
from __future__ import annotations

import argparse

import numpy as np
import torch

from . import inputs, tild


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("workload", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--steps", type=int, default=12)
    ap.add_argument("--flags", type=int, default=0)
    ap.add_argument("--resort-every", type=int, default=0)
    a = ap.parse_args()
    cfg = inputs.CONFIGS[a.workload]
    st = inputs.make_state(cfg)
    eng = tild.Tild(tild.params_from_config(cfg, flags=a.flags, resort_every=a.resort_every))
    d = lambda t: torch.from_numpy(t).cuda()
    eng.tild_set_state(d(st.x), d(st.v), d(st.type), d(st.bond_partner), 0)
    eng.tild_step(a.steps)
    x, v, f, step = eng.tild_get_state(want_v=True, want_f=True)
    e = eng.tild_energy()
    torch.cuda.synchronize()
    x = x.cpu().numpy()
    ok = bool(np.isfinite(x).all() and (x >= 0).all() and (x <= np.array(cfg.box, dtype=np.float32)).all())
    print(f"{cfg.name}: {step} steps, {eng.tild_launch_count()} launches, positions in box: {ok}, "
          f"net force {np.abs(f.cpu().numpy().astype(np.float64).sum(0)).max():.3e}, energies {e}")
    eng.close()


if __name__ == "__main__":
    main()
