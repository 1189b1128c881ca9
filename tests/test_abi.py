"""CPU-only checks of the boundary: the library builds, loads and exports every symbol include/pn.h
declares; the Python options struct matches the C one; the workload generators are deterministic."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_0908_3889_b200 import binding, build

    build.build()
    return binding.load()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "pn.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pn_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    from paper_0908_3889_b200 import binding

    names = declared_functions()
    assert len(names) >= 13
    for n in names:
        assert getattr(lib, n) is not None
    assert sorted(binding.EXPORTS) == names


def test_no_unexpected_dependencies():
    """The product library links only the CUDA runtime and the C/C++ runtime: no oracle, no torch."""
    out = subprocess.check_output(["ldd", os.path.join(ROOT, "paper_0908_3889_b200", "libpn_b200.so")]).decode()
    assert "oracle" not in out and "torch" not in out and "cublas" not in out


def test_options_struct_matches_header(tmp_path):
    from paper_0908_3889_b200.binding import PnOptions

    src = tmp_path / "sz.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "pn.h"\nint main(){printf("%zu %zu %zu %zu %zu",'
                   "sizeof(pn_options), offsetof(pn_options,tau_land), offsetof(pn_options,out_time),"
                   "offsetof(pn_options,stream), offsetof(pn_options,variant));"
                   'printf(" %zu %zu", offsetof(pn_options,hist_bins), offsetof(pn_options,hist_skipped));return 0;}\n')
    exe = tmp_path / "sz"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    got = [int(t) for t in subprocess.check_output([str(exe)]).split()]
    assert got == [C.sizeof(PnOptions), PnOptions.tau_land.offset, PnOptions.out_time.offset,
                   PnOptions.stream.offset, PnOptions.variant.offset, PnOptions.hist_bins.offset, PnOptions.hist_skipped.offset]


def test_new_structs_match_header(tmp_path):
    from paper_0908_3889_b200.binding import PnCheckOut, PnEnsemble, PnStatsOut

    src = tmp_path / "sz2.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "pn.h"\nint main(){printf("%zu %zu %zu %zu %zu %zu %zu",'
                   "sizeof(pn_stats_out), offsetof(pn_stats_out,hist2_norm), sizeof(pn_ensemble), offsetof(pn_ensemble,s1_tilt_deg),"
                   "sizeof(pn_check_out), offsetof(pn_check_out,worst_index), offsetof(pn_check_out,ms_reference));return 0;}\n")
    exe = tmp_path / "sz2"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    got = [int(t) for t in subprocess.check_output([str(exe)]).split()]
    assert got == [C.sizeof(PnStatsOut), PnStatsOut.hist2_norm.offset, C.sizeof(PnEnsemble), PnEnsemble.s1_tilt_deg.offset,
                   C.sizeof(PnCheckOut), PnCheckOut.worst_index.offset, PnCheckOut.ms_reference.offset]


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_0908_3889_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "pn_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, f


def test_status_strings(lib):
    lib.pn_strerror.restype = C.c_char_p
    assert lib.pn_strerror(0) == b"ok"
    assert b"CUDA" in lib.pn_strerror(2)
    assert lib.pn_version() >= 100


def test_workloads_deterministic_and_shaped():
    from paper_0908_3889_b200 import workloads as W

    for name, cfg in W.CONFIGS.items():
        c = W.with_size(cfg, 500)
        y0, m = W.generate(c)
        y1, m1 = W.generate(c)
        assert np.array_equal(y0, y1) and np.array_equal(m, m1)
        assert y0.shape == (500, 10) and m.shape == (500, 2)
        assert np.allclose(m.sum(1), 1.0) and np.all(y0[:, 0] == c.omega0)
        assert np.all(y0[:, 7:10] == [0, 0, 1])
        chi1 = np.linalg.norm(y0[:, 1:4], axis=1) / m[:, 0] ** 2
        chi2 = np.linalg.norm(y0[:, 4:7], axis=1) / m[:, 1] ** 2
        assert chi1.max() <= 1 + 1e-12 and chi2.max() <= 1 + 1e-12
    y0, m = W.generate(W.with_size(W.CONFIGS["C4"], 100))
    assert np.allclose(m, [0.6, 0.4])
    assert np.allclose(y0[:, 1:4], 0.9 * 0.36 * np.array([np.sin(np.pi / 3), 0, 0.5]))
    # isotropy of the sampled directions (mean ~ 0, <z^2> ~ 1/3)
    y0, m = W.generate(W.with_size(W.CONFIGS["C2"], 20000))
    s = y0[:, 4:7] / np.linalg.norm(y0[:, 4:7], axis=1, keepdims=True)
    assert np.abs(s.mean(0)).max() < 0.02 and abs((s[:, 2] ** 2).mean() - 1 / 3) < 0.01
    assert W.CONFIGS["C2"].n == 1 << 20 and W.CONFIGS["C4"].n == 1 << 22 and W.CONFIGS["C5"].n == 1 << 18
