"""SHA-256 of the generator's output, so that a reader can tell that the oracle and the CUDA path saw the same bytes
(BASELINE.md section 3 records these).  `python -m emu_synth.sha256 [--full]`

configs 0-3: the single view of make_config(c) (grains int32 [N,4] little-endian, C order, then view_off int32);
config 4: views 0..15 of the throughput batch (what bench.py's parity leg and the CPU baseline use) and, with --full,
all 1 024 views as bench.py generates them."""
from __future__ import annotations

import hashlib
import sys

import numpy as np

from . import CONFIGS, make_config, make_view


def digest(grains: np.ndarray, view_off: np.ndarray) -> str:
    h = hashlib.sha256()
    h.update(np.ascontiguousarray(grains, "<i4").tobytes())
    h.update(np.ascontiguousarray(view_off, "<i4").tobytes())
    return h.hexdigest()


def config_digest(c: int) -> tuple:
    b = make_config(c)
    return b.n_grains, digest(b.grains, b.view_off)


def batch_digest(first: int, n: int) -> tuple:
    gs = [make_view(CONFIGS[4], 4, v)[0] for v in range(first, first + n)]
    off = np.zeros(n + 1, np.int32)
    off[1:] = np.cumsum([len(g) for g in gs])
    return int(off[-1]), digest(np.concatenate(gs), off)


def main():
    for c in range(4):
        n, d = config_digest(c)
        print(f"config {c}: {n} grains  sha256 {d}")
    n, d = batch_digest(0, 16)
    print(f"config 4, views 0..15: {n} grains  sha256 {d}")
    if "--full" in sys.argv:
        n, d = batch_digest(0, 1024)
        print(f"config 4, views 0..1023: {n} grains  sha256 {d}")


if __name__ == "__main__":
    main()
