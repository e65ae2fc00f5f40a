"""CPU-only checks of the boundary: the C-ABI library builds, loads without a GPU and exports
every symbol include/sft.h declares; the ctypes mirror of sft_plan_desc matches the header; the
binding refuses to run without the library or a device (no CPU fallback)."""
import ctypes
import os
import re
import subprocess
import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "sft.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2502_11823_b200 import build, api
    build.build()
    return api.load_library()


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sft_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_exported(lib):
    from paper_2502_11823_b200 import api
    names = _declared_functions()
    assert {"sft_plan_create", "sft_load_data", "sft_inner_products", "sft_cumulative_snr"} <= set(names)
    for n in names:
        assert hasattr(lib, n), "libsft_b200.so does not export %s" % n
    assert sorted(api.EXPORTS) == names


def test_header_compiles_as_c_and_struct_matches(tmp_path):
    """The header is plain C; offsets of sft_plan_desc printed by a C program equal the ctypes mirror."""
    from paper_2502_11823_b200 import api
    fields = [f[0] for f in api.PlanDesc._fields_]
    prog = ["#include <stdio.h>", "#include <stddef.h>", '#include "sft.h"', "int main(void){",
            'printf("%zu\\n", sizeof(sft_plan_desc));']
    prog += ['printf("%%zu\\n", offsetof(sft_plan_desc, %s));' % f for f in fields]
    prog += ["return 0;}"]
    c = tmp_path / "t.c"
    c.write_text("\n".join(prog))
    exe = tmp_path / "t"
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(c), "-o", str(exe)])
    out = [int(x) for x in subprocess.check_output([str(exe)]).split()]
    assert out[0] == ctypes.sizeof(api.PlanDesc)
    assert out[1:] == [getattr(api.PlanDesc, f).offset for f in fields]


def test_version_and_null_handling(lib):
    assert b"sm_100a" in lib.sft_version()
    assert lib.sft_plan_destroy(None) == 0
    assert lib.sft_plan_create(None, None) == 1           # SFT_EINVAL
    assert b"NULL" in lib.sft_last_error(None)
    assert lib.sft_plan_launch_count(None) == 0


def test_argument_validation_before_any_device_use(lib):
    """Descriptor errors are reported as status codes + message (never an exception/abort)."""
    from paper_2502_11823_b200 import api
    base = dict(n_channels=1, n_sft=8, t_sft=8.0, fs=512.0, k_lo=10, k_hi=50, K=4, f_ref=20.0, f_hi=30.0)
    for bad, code in [(dict(n_channels=0), "SFT_EINVAL"), (dict(n_channels=5), "SFT_EINVAL"),
                      (dict(t_sft=8.001), "SFT_ESHAPE"), (dict(k_hi=10), "SFT_ESHAPE"),
                      (dict(K=1000), "SFT_EINVAL"), (dict(f_ref=0.0), "SFT_EINVAL"),
                      (dict(kernel=7), "SFT_EINVAL"), (dict(n_sft=0), "SFT_EINVAL")]:
        with pytest.raises(api.SftError) as ei:
            api.Plan(dict(base, **bad))
        assert code in str(ei.value), (bad, str(ei.value))


def test_no_cpu_fallback_without_device(lib):
    """Without a CUDA device plan creation fails loudly (SFT_ECUDA / SFT_EINVAL), it never computes on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2502_11823_b200 import api
    with pytest.raises(api.SftError):
        api.Plan(dict(n_channels=1, n_sft=8, t_sft=8.0, fs=512.0, k_lo=10, k_hi=50, K=4, f_ref=20.0, f_hi=30.0))


def test_product_path_does_not_import_oracle():
    """The package never imports oracle/ (parity rule): checked on the source text."""
    pkg = os.path.join(ROOT, "paper_2502_11823_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "_work/" not in txt, f


def test_binding_rejects_wrong_dtypes(lib):
    from paper_2502_11823_b200 import api
    with pytest.raises(TypeError):
        api._ptr(np.zeros(4, np.float32), np.float64, (4,), "x")
    with pytest.raises(ValueError):
        api._ptr(np.zeros(4, np.float64), np.float64, (5,), "x")
    with pytest.raises(TypeError):
        api._ptr(np.zeros((4, 4), np.float64)[:, ::2], np.float64, None, "x")


def test_tsft_rule_against_the_papers_tables():
    """sft_tsft_rule (host arithmetic, no device): Eq.(34) P:248 reproduces the paper's printed Table I within 2 % with this
    library's PN waveform (the paper uses IMRPhenomT), max fddot ~ 5e-6 Hz/s^2, the delta^(1/3) law of Table II
    exactly, and Table II itself within 6 % at 0PN (the 1PN expansion is poor that close to MECO)."""
    import json
    import os
    from paper_2502_11823_b200 import api
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))
    eta, mc = 0.25, 2.8 * 0.25 ** 0.6
    for pn1 in (0, 1):
        for d, T in zip(g["table1"]["delta"], g["table1"]["t_sft"]):
            t, fdd = api.tsft_rule(mc, eta, 10.0, d, pn1)
            assert abs(t - T) <= 0.02 * T, (pn1, d, t, T)
            assert abs(fdd - g["bns"]["max_fddot_printed"]) <= 0.05 * g["bns"]["max_fddot_printed"]
    mc2 = 2e6 * 0.25 ** 0.6
    ts = [api.tsft_rule(mc2, eta, 1.9e-3, d, 0)[0] for d in g["table2"]["delta"]]
    for d, t, T in zip(g["table2"]["delta"], ts, g["table2"]["t_sft"]):
        assert abs(t - T) <= 0.06 * T, (d, t, T)
        assert abs(t / ts[0] - (d / g["table2"]["delta"][0]) ** (1.0 / 3.0)) < 1e-12
    import pytest
    with pytest.raises(api.SftError):
        api.tsft_rule(mc, 0.3, 10.0, 1.0)
