"""Writes the stored oracle trajectories under tests/golden/.  Calls ONLY oracle/ and the input generator.

    python tests/golden/make_golden.py cfg0 cfg1 ...

The paper prints no expected values, so these fixtures are oracle outputs, not paper numbers: the
(sweep, F, theta) history of Algorithm 1 on the named BASELINE.json config, produced by
oracle.fix on the gf_inputs field.  They exist because the full-size oracle runs take minutes to hours on host cores;
the GPU parity tests compare the CUDA path's history with them (F rel 1e-10 / 1e-5, theta within x1.5, sweep count
+-2 %).  FP32 configs follow reading A18: the FP64 oracle is fed the FP32-rounded input with 12-real emulation.
"""
import json
import os
import sys
import time

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import gf_inputs as gi  # noqa: E402
import oracle  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))


def run(cfg):
    dims = cfg["dims"]
    U = gi.make_links(dims, cfg["roughness"], cfg["seed"], dtype=np.float32 if cfg["prec"] == "f32" else np.float64)
    U = np.ascontiguousarray(U.astype(np.float64))
    if cfg["storage"] == 12:
        oracle.project12(U, dims)
    t = time.time()
    done, hist = oracle.fix(U, dims, cfg["gauge"], cfg["omega"], cfg["eps"], cfg["max_sweeps"], cfg["check_every"],
                            cfg["reunit_every"], cfg["storage"])
    out = dict(config={k: (list(v) if isinstance(v, tuple) else v) for k, v in cfg.items()},
               citation="oracle.fix = Algorithm 1, PAPER.md:70-95; F, theta = eqs. 1.1-1.3, PAPER.md:20-33",
               written_by="tests/golden/make_golden.py (oracle only)", sweeps_done=done,
               history=[[int(s), repr(float(F)), repr(float(th))] for s, F, th in hist],
               oracle_seconds=round(time.time() - t, 1), threads=oracle.num_threads())
    with open(os.path.join(HERE, f"{cfg['name']}_trajectory.json"), "w") as f:
        json.dump(out, f, indent=1)
    print(cfg["name"], "sweeps", done, "F", hist[-1, 1], "theta", hist[-1, 2], f"{time.time() - t:.1f}s", flush=True)


if __name__ == "__main__":
    names = sys.argv[1:] or ["cfg0"]
    for c in gi.CONFIGS:
        if c["name"] in names:
            run(c)
