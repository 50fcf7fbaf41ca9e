"""Sensitivity loss of the nearest-bin (zero-padding) approximation against exact pointing, as a function of the
padding factor P ("a padding factor of P = 2 has been chosen"; Fig. 1).

For every coarse channel and every N-S beam the clamped bin J (oracle.ns_index, eq. (1)+(2)) misses the desired
pointing by d = turns - J / NP cycles per feed; a point source at the desired pointing is then received with the
power fraction (sin(pi N d) / (N sin(pi d)))^2 of the Dirichlet kernel (pinned by P3 / P15c).  The table gives, over
the 1024 channels x 256 beams, the mean and worst loss 1 - fraction, for beams inside the alias-free range
|turns| < 1/2.  Test infrastructure: calls only oracle/.  Writes tests/golden/beam_loss_vs_padding.json.

    python oracle/beam_loss_table.py
"""
import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import oracle  # noqa: E402


def loss_table(pads=(1, 2, 4), n_chan=1024):
    out = {}
    for P in pads:
        NP = 256 * P
        losses = []
        for k in range(n_chan):
            f = 800.0 - k * 0.390625
            turns = oracle.ns_turns(f)
            J = oracle.ns_index(f, NP).astype(np.float64)
            d = turns - J / NP
            d -= np.rint(d)
            inside = np.abs(turns) < 0.5
            with np.errstate(invalid="ignore", divide="ignore"):
                frac = np.where(d == 0, 1.0, (np.sin(np.pi * 256 * d) / (256 * np.sin(np.pi * d))) ** 2)
            losses.append(1.0 - frac[inside])
        a = np.concatenate(losses)
        out[str(P)] = {"zero_pad": NP, "mean_loss": float(a.mean()), "worst_loss": float(a.max()),
                       "p95_loss": float(np.quantile(a, 0.95)), "n_beams": int(a.size)}
    return out


if __name__ == "__main__":
    tab = loss_table()
    path = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "tests", "golden",
                        "beam_loss_vs_padding.json")
    with open(path, "w") as f:
        json.dump({"source": "oracle/beam_loss_table.py (oracle.ns_index, oracle.ns_turns; Dirichlet closed form)",
                   "cite": "PAPER.md:61 (padding factor trade-off), :63-65 (Fig. 1), :98 (beam interpolation)",
                   "loss_by_padding_factor": tab}, f, indent=1)
    for P, r in tab.items():
        print(f"P = {P}: mean loss {100 * r['mean_loss']:.2f} %, 95th percentile {100 * r['p95_loss']:.2f} %, "
              f"worst {100 * r['worst_loss']:.2f} %  ({r['n_beams']} beams)")
