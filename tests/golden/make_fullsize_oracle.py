#!/usr/bin/env python
"""Writes tests/golden/fullsize_oracle.json: what the float64 ORACLE reaches on BASELINE.json's
configs[2] and configs[3] at their stated sizes and iteration counts.

    python tests/golden/make_fullsize_oracle.py            (about 25 minutes on 8 cores)

Calls only ``oracle/`` and ``workloads/`` (the seeded input generators); nothing here touches the CUDA
path.  tests/test_gpu_fullsize.py compares the CUDA library's fits of the SAME initial sets (which the
test regenerates through the oracle's own initialiser and checks against the SHA-256 stored here)
against these values: PSNR within 0.05 dB, loss within 2 %, selected counts within 2 % of N
(north_star tolerances; PAPER.md:57, 64 I-frame optimisation steps, PAPER.md:90-94 P-frame refit).

  configs[2]: 1920x1080 frame 0 of SPEC_1080P, 50,000 Gaussians from init_roi(seed 1, scales [1,8]),
              2,000 iterations, lr 1e-2: loss trace every 100 iterations, final loss and PSNR.
  configs[3]: 1920x1080 frames 0..3 of SPEC_PSEQ (head +2 px and +0.5 deg per frame, fresh noise):
              frame 0 as an I-frame (init_roi seed 3, 2,000 iterations), then three P-frames of 200
              iterations each on the Gaussians the tile-residual rule selects at tau = 0.02.
"""
import hashlib
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import workloads as wl  # noqa: E402

W, H, N = 1920, 1080, 50_000
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "fullsize_oracle.json")


def init_hash(mu, chol, rgb, op) -> str:
    h = hashlib.sha256()
    for a in (mu, chol, rgb, op):
        h.update(np.ascontiguousarray(a, dtype=np.float32).tobytes())
    return h.hexdigest()


def main():
    res = {"written_by": "tests/golden/make_fullsize_oracle.py (oracle/ only)", "W": W, "H": H, "N": N, "lr": 1e-2,
           "threads": oracle.get_threads()}
    t0 = time.time()

    # ---- configs[2]
    frame, mask = wl.talking_head_frame(wl.SPEC_1080P, 0)
    mu, chol, rgb, op, _ = oracle.init_roi(frame, mask, N, 1, 1.0, 8.0)
    p = oracle.Params.from_f32(wl.GaussianSet(mu, chol, rgb, op))
    rep = oracle.fit(W, H, p, frame, 2000, lr=1e-2, trace=True)
    res["config2"] = {"init_seed": 1, "init_sha256": init_hash(mu, chol, rgb, op), "iters": 2000,
                      "final_loss": rep.final_loss, "psnr": rep.psnr,
                      "loss_trace_every_100": [float(x) for x in rep.loss_trace[::100]]}
    print("config2", rep.psnr, rep.final_loss, time.time() - t0, flush=True)

    # ---- configs[3]
    frames = [wl.talking_head_frame(wl.SPEC_PSEQ, k) for k in range(4)]
    mu, chol, rgb, op, _ = oracle.init_roi(frames[0][0], frames[0][1], N, 3, 1.0, 8.0)
    p = oracle.Params.from_f32(wl.GaussianSet(mu, chol, rgb, op))
    rep = oracle.fit(W, H, p, frames[0][0], 2000, lr=1e-2)
    seq = {"init_seed": 3, "init_sha256": init_hash(mu, chol, rgb, op), "tau": 0.02, "iframe_iters": 2000,
           "pframe_iters": 200, "iframe": {"final_loss": rep.final_loss, "psnr": rep.psnr}, "pframes": []}
    print("config3 I", rep.psnr, time.time() - t0, flush=True)
    for k in (1, 2, 3):
        act, r = oracle.encode_pframe(W, H, p, frames[k][0], 0.02, 200, lr=1e-2)
        seq["pframes"].append({"frame": k, "n_active": int(r.n_active), "iters_run": int(r.iters_run),
                               "final_loss": r.final_loss, "psnr": r.psnr})
        print("config3 P", k, r.n_active, r.psnr, time.time() - t0, flush=True)
    res["config3"] = seq
    res["seconds"] = time.time() - t0
    with open(OUT, "w") as f:
        json.dump(res, f, indent=1)
        f.write("\n")


if __name__ == "__main__":
    main()
