"""Runs the fp32 oracle on BASELINE config 3 for its full 1000 steps with its FTZ/DAZ switch on, in a process of its own,
and writes the ten final arrays to a directory (fp32 .npy).  Test infrastructure (calls only oracle/ and the input
generators).  A process of its own because the oracle sets the flush bits in the MXCSR of its OpenMP workers and never
clears them, and the other parity tests need the oracle in plain IEEE arithmetic; with the flush on because 1000 steps at
552^3 in IEEE arithmetic spend 2.5x as long in denormal assists (16 min on the test box's Xeon cores)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from oracle import Oracle  # noqa: E402
from paper_2606_06910_b200 import inputs  # noqa: E402


def main(out_dir):
    w = inputs.config(3)
    o = Oracle(w.n_interior, w.cpml, **w.cpml_kwargs())
    o.set_model(w.c)
    o.set_sources(w.sources, w.wavelets)
    o.set_ftz(True)
    oracle.set_threads(oracle.max_threads())
    o.step(w.steps)
    for i in range(10):
        np.save(os.path.join(out_dir, "a%d.npy" % i), o.get(i).astype(np.float32))     # lossless: the fp32 instantiation
    o.close()


if __name__ == "__main__":
    main(sys.argv[1])
