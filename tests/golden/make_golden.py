"""Writes tests/golden/full_size.json: SHA-256 of the CPU oracle's outputs on the five full-size
BASELINE.json configurations and on the 3 M-point parity case (plus the SHA-256 of the generated
inputs, to catch generator drift).

Calls ONLY ``oracle`` and the seeded input generators -- never the CUDA path.  The GPU parity test
compares the CUDA outputs' hashes with these (a hash of the whole array is a bit-exact comparison
of every element).

  python tests/golden/make_golden.py [C1 C2 ... L3M]            squared distance: oracle.fps        -> key "C5"
  python tests/golden/make_golden.py --euclid [C4 C5 ...]       Euclidean mode:   oracle.fps_euclid -> key "C5:euclid"
"""
import fcntl
import hashlib
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from paper_2606_06255_b200 import inputs  # noqa: E402

OUT = os.path.join(HERE, "full_size.json")


def sha(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


def main(names, euclid):
    fn = oracle.fps_euclid if euclid else oracle.fps
    for name in names:
        w = inputs.WORKLOADS.get(name) or inputs.EXTRA_WORKLOADS[name]
        P = inputs.make_batch(w)
        t = time.time()
        idx, mind = fn(P, w.M, w.start_idx)
        dt = time.time() - t
        rec = {
            "B": w.B, "N": w.N, "M": w.M, "start_idx": w.start_idx, "seed": inputs.BASE_SEED,
            "input_sha256": sha(P), "idx_sha256": sha(idx.astype(np.int32)), "mindist_sha256": sha(mind.astype(np.float32)),
            "idx_head": idx.reshape(w.B, w.M)[0, :8].tolist(),
            "mindist_tail_bits": [int(v) for v in mind.reshape(w.B, w.M)[0, -4:].view(np.uint32)],
            "oracle_seconds": round(dt, 2),
            "written_by": "tests/golden/make_golden.py (%s only)" % ("oracle/fps_oracle_euclid.c" if euclid else "oracle/fps_oracle.c"),
        }
        if not euclid:
            rec["oracle_threads"] = int(oracle.fps.threads_used)
        print(name, rec, flush=True)
        # several instances may run side by side (the large cases take minutes each): read-modify-write under a lock
        with open(OUT + ".lock", "w") as lk:
            fcntl.flock(lk, fcntl.LOCK_EX)
            data = json.load(open(OUT)) if os.path.exists(OUT) else {}
            data[name + (":euclid" if euclid else "")] = rec
            json.dump(data, open(OUT, "w"), indent=1, sort_keys=True)


if __name__ == "__main__":
    args = sys.argv[1:]
    euclid = "--euclid" in args
    args = [a for a in args if a != "--euclid"]
    main(args or ["C1", "C2", "C3", "C4", "C5"], euclid)
