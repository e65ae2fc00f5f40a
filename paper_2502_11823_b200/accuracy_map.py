"""Accuracy maps r(delta, Delta k) of section IV (Eq.(36); Fig. 3, Fig. 4) on the GPU path.

    python -m paper_2502_11823_b200.accuracy_map --example bns|mbhb [--deltas ...] [--dks ...] [--dc 0|1]

For each delta the SFT length follows from the library's own rule (``sft_tsft_rule``, Eq.(34)); the noiseless fiducial
signal of the example (``workloads.accuracy_case``: the paper's masses, band, sampling rate and projector, with this library's
PN waveform in place of IMRPhenomT) is turned into data SFTs on the device (``sft_ingest_timeseries``), and ([d,h]) of the
fiducial template (``sft_inner_products``, band half-width K = Delta k / 2) is compared with <d,h> "by direct integration"
(the time-domain sum (2 dt / S) sum_j h_j^2, computed here on the host) through r = 1 - sqrt(([d,h]) / <d,h>).
One JSON line per (delta, Delta k).  ``--dc 1`` lets the bin k = 0 count (``include_dc``): the paper's sums do, and
the massive-BBH example lives below the first bin for most of its duration (edge effects, section IV.D).
The exact values of the paper's colour maps are not reproduced (different waveform model); their magnitudes are
(tests/test_gpu_accuracy.py, profiles/).
"""
import argparse
import json
import sys

import numpy as np

from . import api, workloads as wl

PAPER_DELTAS = {"bns": (3.0, 2.5, 2.0, 1.5, 1.0, 0.5), "mbhb": (1.0, 0.5, 0.25, 0.1, 0.05, 0.01)}   # Table I, Table II


def t_sft_for(example, delta, pn1=1):
    """SFT length of Eq.(34) for the example's masses and final frequency."""
    m1, m2, _, f1, _, _ = wl.ACCURACY_EXAMPLES[example]
    eta = m1 * m2 / (m1 + m2) ** 2
    return api.tsft_rule((m1 + m2) * eta ** 0.6, eta, f1, delta, pn1)[0]


def accuracy_point(example, delta, dk, include_dc=0, f_start=None, pn1=1, device=0):
    """r of Eq.(36) for one (delta, Delta k).  Returns a dict."""
    K = max(0, int(dk) // 2)
    w = wl.accuracy_case(example, t_sft_for(example, delta, pn1), K, f_start=f_start, pn1=pn1)
    d = dict(w.desc, include_dc=int(include_dc), evaluator="direct")        # one template: no point in building tables
    with api.Plan(d, device=device) as plan:
        plan.ingest_timeseries(0, np.ascontiguousarray(w.series[0]), np.ascontiguousarray(w.psd_scale[0]),
                               np.ascontiguousarray(w.psd_shape[0]), np.ascontiguousarray(w.response[0]))
        xh, hh = np.empty(1), np.empty(1)
        plan.inner_products(np.ascontiguousarray(w.params), xh, hh)
    exact = w.notes["xx_time"]
    ratio = xh[0] / exact
    return dict(example=example, delta=float(delta), delta_k=2 * K, t_sft=w.desc["t_sft"], n_sft=w.desc["n_sft"],
                include_dc=int(include_dc), r=(1.0 - np.sqrt(ratio)) if ratio >= 0 else None, ratio=float(ratio),
                xh=float(xh[0]), hh=float(hh[0]), exact=float(exact))


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--example", default="bns", choices=sorted(wl.ACCURACY_EXAMPLES))
    ap.add_argument("--deltas", type=float, nargs="*", default=None)
    ap.add_argument("--dks", type=int, nargs="*", default=(2, 4, 10, 20, 50, 100, 200))
    ap.add_argument("--dc", type=int, default=None, help="include the k = 0 bin (default: 1 for mbhb, 0 for bns)")
    ap.add_argument("--f-start", type=float, default=None, dest="f_start")
    a = ap.parse_args(argv)
    dc = a.dc if a.dc is not None else int(a.example == "mbhb")
    for delta in (a.deltas or PAPER_DELTAS[a.example]):
        for dk in a.dks:
            print(json.dumps(accuracy_point(a.example, delta, dk, dc, a.f_start)), flush=True)


if __name__ == "__main__":
    sys.exit(main())
