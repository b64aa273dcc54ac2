"""The setup-time scheduler (csrc/plan.cpp: ~1,100 lines of index arithmetic) under AddressSanitizer,
UndefinedBehaviorSanitizer and LeakSanitizer: plans for all five configs, a 70-sibling star, odd offsets and a
20,000-compartment root branch with a fork, under fourteen option sets (fp32, no grouping, level-mean and block-mean splitting,
factored, small segments / chunks / clusters, split items, streaming, no cable path).  Host only, no GPU needed."""
import os
import shutil
import subprocess

import numpy as np
import pytest

import morphgen as mg
from helpers import random_parent

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.skipif(shutil.which("g++") is None, reason="g++ not available")
def test_plan_create_under_asan_ubsan(tmp_path):
    cases = []
    for cfg, scale in ((0, 1.0), (1, 0.005), (2, 0.01), (3, 0.005), (4, 1.0)):
        m = mg.make_config(cfg, scale)
        cases.append((m.parent, m.cell_offsets))
    star = np.array([-1] + [0] * 70, np.int32)
    ps = [star, random_parent(33, 1), np.array([-1], np.int32), random_parent(200, 2, .7), star[:40], random_parent(1001, 3, .97)]
    cases.append((np.concatenate(ps), np.concatenate([[0], np.cumsum([len(p) for p in ps])])))
    n = 20000
    p = np.arange(-1, n + 1, dtype=np.int32); p[n + 1] = n - 1
    cases.append((p, np.array([0, n + 2])))
    for k, (par, offs) in enumerate(cases):
        np.asarray(par, np.int32).tofile(tmp_path / f"p{k}.bin")
        np.asarray(offs, np.int64).tofile(tmp_path / f"o{k}.bin")
    exe = str(tmp_path / "drv")
    csrc = os.path.join(ROOT, "paper_1810_12742_b200", "csrc")
    subprocess.check_call(["g++", "-std=c++17", "-O1", "-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer",
                           "-I", os.path.join(ROOT, "include"), "-I", csrc, os.path.join(ROOT, "tests", "asan_plan_driver.cpp"),
                           os.path.join(csrc, "plan.cpp"), "-o", exe])
    r = subprocess.run([exe, str(len(cases)), str(tmp_path)], capture_output=True, text=True, timeout=600,
                       env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1", UBSAN_OPTIONS="print_stacktrace=1"))
    out = r.stdout + r.stderr
    assert r.returncode == 0, out[-3000:]
    assert "AddressSanitizer" not in out and "runtime error" not in out and "LeakSanitizer" not in out, out[-3000:]
    assert f"plans built under ASan/UBSan: {14 * len(cases)}" in out
