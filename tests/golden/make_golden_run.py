"""Writes tests/golden/run_cfg<k>.npz: the ORACLE's forward + adjoint run of BASELINE.json configs[k] on the
seeded inputs of paper_2211_09815_b200.inputs, sampled at a fixed random subset of particles.

    python tests/golden/make_golden_run.py 1        # ~25 min on 8 cores for configs[1]

Calls only oracle/ and the input generators -- never the CUDA path.  The GPU parity test at full size
(tests/test_gpu_full_size.py) compares against these stored oracle values.
Stored: J, idx[S] (particle ids, default_rng(7)), and s_n, p_n, xi0, pi0, dJ_ds0 at idx (float64).
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import pm_oracle as orc  # noqa: E402
from paper_2211_09815_b200 import inputs  # noqa: E402

N_SAMPLE = 16384


def golden_inputs(k):
    """The seeded inputs of configs[k] (shared recipe: DESIGN.md 'Input recipe').  p0 needs G_D/D1 at a_0,
    a host scalar: the caller passes it (the oracle's here, libpm's own in bench.py)."""
    cfg = inputs.config(k)
    s0 = inputs.zeldovich_displacement(cfg["lattice"], cfg["mesh"], seed=1, rms=0.3)
    target = inputs.lognormal_target(cfg["mesh"], seed=2, sigma=1.0)
    return cfg, s0, target


def main(k):
    cfg, s0, target = golden_inputs(k)
    ratio = orc.p_over_s(cfg["omega_m"], cfg["a"][0])
    p0 = (s0.astype(np.float64) * ratio).astype(np.float32)
    t = time.time()
    out = orc.run_fwd_adj(cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"], s0, p0, target)
    dt = time.time() - t
    npart = s0.shape[0]
    idx = np.sort(np.random.default_rng(7).choice(npart, size=min(N_SAMPLE, npart), replace=False))
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"run_cfg{k}.npz")
    np.savez_compressed(path, J=out["J"], idx=idx, p_over_s=ratio, oracle_seconds=dt, threads=orc.num_threads(),
                        **{key: out[key][idx] for key in ("s_n", "p_n", "xi0", "pi0", "dJ_ds0", "s_rec", "p_rec")})
    print(f"wrote {path}: J = {out['J']:.10e}, oracle {dt:.0f} s on {orc.num_threads()} threads")


if __name__ == "__main__":
    main(int(sys.argv[1]) if len(sys.argv) > 1 else 1)
