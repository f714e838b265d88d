"""Writes tests/golden/config_samples_<name>.npz: sampled outputs of the FULL BASELINE configurations computed by
the CPU oracle (and nothing else).  Run from the repo root:

    python tests/golden/make_config_goldens.py config2 config3 config4

Each file holds, for the named configuration at its full size and step count: the dt of every cycle, 4096 seeded
sample points (flat cell indices) and, at those points, the 5 conserved variables and the 3 face-field components
after the last cycle, plus per-field max|.| (for the relative-error norm) and the field sums.
Only oracle/ and the seeded input generators are imported; no value comes from the CUDA path.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import idfxref  # noqa: E402
from paper_2304_13746_b200 import inputs  # noqa: E402

NSAMPLES = 4096


def sample_indices(n, seed):
    rng = np.random.Generator(np.random.PCG64(seed + 77))
    return np.sort(rng.choice(n ** 3, size=NSAMPLES, replace=False))


def main(names):
    for name in names:
        prim, b, cfg = inputs.make(name)
        n = cfg["n"]
        o = idfxref.Oracle(n, n, n, cfg["dx"], cfg["gamma"], cfg["solver"], cfg["limiter"], cfg["emf"])
        o.set_state(prim.numpy(), None if b is None else b.numpy())
        dts = []
        t0 = time.time()
        for s in range(cfg["steps"]):
            assert o.advance(1, cfg["cfl"]) == 0
            dts.append(o.last_dt())
            print(name, "step", s + 1, "/", cfg["steps"], "dt", dts[-1], "%.0fs" % (time.time() - t0), flush=True)
        cons, bf = o.get_conserved()
        idx = sample_indices(n, cfg["seed"])
        out = dict(n=n, steps=cfg["steps"], dts=np.array(dts), idx=idx,
                   cons=cons.reshape(5, -1)[:, idx], cons_max=np.abs(cons).reshape(5, -1).max(1),
                   cons_sum=cons.reshape(5, -1).sum(1), roe_fallbacks=o.roe_fallbacks())
        if bf is not None:
            out.update(bface=bf.reshape(3, -1)[:, idx], bface_max=np.abs(bf).max(), bface_sum=bf.reshape(3, -1).sum(1))
        np.savez(os.path.join(os.path.dirname(os.path.abspath(__file__)), "config_samples_%s.npz" % name), **out)


if __name__ == "__main__":
    main(sys.argv[1:] or ["config2", "config3", "config4"])
