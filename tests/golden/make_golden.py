"""Writes tests/golden/config1_oracle.txt from the ORACLE ONLY (never from the CUDA path).

The paper prints no worked numeric example, so this fixture is not a pin of the
oracle against the paper; it freezes the oracle's own output on BASELINE.json configs[0] (1 event, 20
tracks, seed 1) so that any later change to the oracle's arithmetic shows up as a diff that the commit
message has to justify.  Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle   # noqa: E402
import synth    # noqa: E402


def main():
    geom, b, p = synth.make_workload(1)
    h, t = oracle.run_batch(b, geom, p)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_oracle.txt")
    with open(out, "w") as f:
        f.write("# oracle output on BASELINE.json configs[0]; written by tests/golden/make_golden.py (oracle only)\n")
        f.write(f"# n_hits {h.n_hits}\n")
        f.write("# hits: index id x_at_y0(hex f32)\n")
        for k in range(h.n_hits):
            f.write(f"H {k} {int(h.id[k])} {h.x_at_y0[k:k+1].view(np.uint32)[0]:08x}\n")
        f.write("# tracks: t n_hits h0 h1 h2 h3 qop(hex f32) chi2(hex f32)\n")
        for k in range(b.n_velo_total):
            f.write(f"T {k} {int(t.n_hits[k])} " + " ".join(str(int(v)) for v in t.hit_idx[:, k]) +
                    f" {t.qop[k:k+1].view(np.uint32)[0]:08x} {t.chi2[k:k+1].view(np.uint32)[0]:08x}\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
