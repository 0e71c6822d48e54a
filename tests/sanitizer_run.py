"""Small solves for compute-sanitizer (race detection row): configs 1-2 at reduced size and one masked + hoisted
case, each through the persistent kernel and through the per-kernel launches, with the result checked against the oracle so that
a run that "passes" the tool is also known to have computed the right thing.

    compute-sanitizer --tool memcheck|racecheck|synccheck|initcheck python tests/sanitizer_run.py

Not collected by pytest (no test_ prefix); profiles/r2_sanitizer.md records the runs.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import torch  # noqa: E402
from oracle import oracle  # noqa: E402
from paper_1306_2461_b200 import binding as B, synthetic as syn  # noqa: E402
from parity import assert_parity  # noqa: E402


def run(c, persistent, mask=None, hoist=False, fused=True):
    ref = oracle.solve(c.I1, c.I2, c.levels, c.window_radius, c.iterations, c.window_type, mask=mask)
    with B.OpticalFlow(*c.create_args) as of:
        of.set_persistent(persistent)
        of.set_fused(fused)
        of.set_hoist(hoist)
        if mask is not None:
            of.set_mask(mask)
        d1 = torch.from_numpy(c.I1.view(np.int16) if c.I1.dtype == np.uint16 else c.I1).cuda()
        d2 = torch.from_numpy(c.I2.view(np.int16) if c.I2.dtype == np.uint16 else c.I2).cuda()
        for _ in range(2):                                   # twice: barrier word and ring parity carry over
            u, v = of.compute(d1, d2)
        m = of.validity()
        torch.cuda.synchronize()
        st = assert_parity(u.cpu().numpy(), v.cpu().numpy(), m.cpu().numpy(), ref, c.name)
    print("ok", c.name, c.width, c.height, "persistent" if persistent else "per-kernel", "mask" if mask is not None else "", "hoist" if hoist else "",
          "fused" if fused else "two-pass", st, flush=True)


def main():
    oracle.build()
    c1 = syn.config1()                                       # 256x256, 1 level, box R=8, 4 iterations (fused level 0)
    c2 = syn.config2(448, 320)                               # config 2 at reduced size: 2 levels, box R=7, 6 iterations
    c3 = syn.config3(320, 256)                               # 3 levels, Gaussian R=12
    mask = syn.mask_backward_step(320, 256)
    for persistent in (True, False):
        run(c1, persistent)
        run(c2, persistent)
    run(c2, True, fused=False)                               # two-pass form at every level inside the persistent kernel
    run(c3, True, mask=mask, hoist=True)
    run(c3, False, mask=mask, hoist=True)
    print("sanitizer_run: all cases ok")


if __name__ == "__main__":
    main()
