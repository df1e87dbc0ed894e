"""Writes tests/golden/oracle_samples_cfg{4,5}.npz: sampled entries of the ORACLE's projection of the full-size
BASELINE.json configs whose blocks take the oracle minutes (n = 2401 of config 4, n = 4096 of config 5).

Calls only oracle/ and the seeded input generators (workloads/); nothing here touches the CUDA path.  The GPU
parity tests compare the library's output at the same svec indices (tests/test_gpu_parity.py), so that the
full-size comparison against the oracle itself does not need an hour of host time on the GPU box.

    python tests/golden/make_oracle_samples.py [5] [4]

Stored per config: `idx` (svec indices: a fixed stride plus every diagonal entry), `val` (oracle output there),
`norm` (2-norm of the whole oracle output), `in_norm`, `seconds`, `threads`.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle      # noqa: E402
import workloads   # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))


def sample_indices(sizes, stride=4099):
    total = sum(n * n for n in sizes)
    idx = set(range(0, total, stride))
    off = 0
    for n in sizes:
        for j in range(n):
            idx.add(off + j * (2 * n - j))          # diagonal entry X_jj (start of column j)
        off += n * n
    return np.array(sorted(idx), dtype=np.int64)


def main():
    cfgs = [int(a) for a in sys.argv[1:]] or [5, 4]
    oracle.build()
    for cfg in cfgs:
        w = workloads.make(cfg)
        sv = np.concatenate([oracle.pack(b.X) for b in w.blocks])
        t0 = time.perf_counter()
        out = oracle.project(w.sizes, sv, nthreads=oracle.max_threads())
        dt = time.perf_counter() - t0
        idx = sample_indices(w.sizes)
        np.savez_compressed(os.path.join(HERE, f"oracle_samples_cfg{cfg}.npz"), idx=idx, val=out[idx],
                            norm=np.linalg.norm(out), in_norm=np.linalg.norm(sv), seconds=dt, threads=oracle.max_threads())
        print(f"cfg{cfg}: {len(idx)} samples, oracle {dt:.1f} s on {oracle.max_threads()} threads, ||out|| = {np.linalg.norm(out):.6f}")


if __name__ == "__main__":
    main()
