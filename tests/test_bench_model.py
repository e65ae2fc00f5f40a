"""Host logic of bench.py: the instruction-count models behind roofline.frac and the files it cites."""
import os
import re
import types

import numpy as np

import bench

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _w(K=8, C=1, name="config2-F"):
    return types.SimpleNamespace(desc=dict(K=K, n_channels=C), name=name)


def test_counts_are_ordered_and_mix_weighted():
    """strict <= current kernel's count <= fixed count on the table paths; the line's figures are the path-mix averages."""
    for K, C in ((8, 1), (16, 2), (4, 1)):
        for path in ("table", "table2", "fresnel", "series1", "series3"):
            fixed = bench.alg_instr_per_pair(path, K, C)
            kern = bench.kernel_instr_per_pair(path, K, C)
            strict = bench.kernel_instr_per_pair(path, K, C, strict=True)
            assert 0 < strict < kern <= fixed, (path, K, C)
    paths = dict(series0=0, series1=0, series2=0, series3=0, fresnel=106496, table=39080960, table2=626688)   # config 2-F
    r = bench.roofline(_w(), 39813120, 0.2588, paths, "auto", dict(ffma=34700.0, table_mix_ipc=0.9))
    assert abs(r["alg_instr_per_pair"] - 149.42) < 0.05
    assert r["frac_strict"] < r["frac_kernel_count"] < r["frac"] < r["frac_of_measured_ffma_issue"] < r["frac_of_mix_ceiling"] < 1.0
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and abs(r["peak"] - 148 * 4 * 32 * 1.965) < 1e-9
    assert abs(r["frac"] - 0.618) < 0.003                       # the committed line (profiles/r02_bench.json.txt)
    assert abs(r["kernel_instr_per_pair"] - 117.5) < 0.5        # 112.5 on the common path (225 SASS instructions per two SFTs), path-mix average
    assert bench.roofline(_w(), 1, None, paths) is None and bench.roofline(_w(), 1, 0.1, None) is None


def test_traffic_figures_cite_committed_captures():
    for (wname, ev), (bytes_, src) in bench.NCU_TRAFFIC.items():
        assert bytes_ > 0 and os.path.exists(os.path.join(ROOT, src)), src
    txt = open(os.path.join(ROOT, "profiles", "r02_main_kernel.md")).read()
    m = re.search(r"`dram__bytes_read.sum` \| Mbyte \| ([0-9.]+)", txt)
    assert m and abs(float(m.group(1)) * 1e6 - bench.NCU_TRAFFIC[("config2-F", "auto")][0]) < 2e5
