"""the CPU oracle built under -fsanitize=address,undefined runs the whole chain
(R0..R6, refit, merging, three-iteration fit) on a small full-TPC frame without a report."""
import os
import subprocess

import numpy as np

from paper_2601_20569_b200 import datagen as dg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    src = [os.path.join(ROOT, "oracle", f) for f in ("sanitize_driver.cpp", "tpc_oracle.cpp", "tpc_merge_oracle.cpp",
                                                       "tpc_fit_oracle.cpp")]
    exe = str(tmp_path / "oracle_asan")
    subprocess.run(["g++", "-O1", "-g", "-std=c++17", "-ffp-contract=off", "-fsanitize=address,undefined",
                    "-fno-sanitize-recover=undefined", "-pthread", *src, "-o", exe], check=True)
    cl, _, _ = dg.generate(dg.preset("C2", tracks_per_event=400, seed=5))
    # plus what the edge-case tests feed: NaN / Inf coordinates, clusters outside the acceptance, a bad row
    extra = np.zeros(4, dtype=cl.dtype)
    extra["row"] = [10, 10, 200, 11]
    extra["y"] = [np.nan, 500.0, 0.0, 0.0]
    extra["z"] = [1.0, 2.0, 3.0, np.inf]
    cl = np.concatenate([cl, extra])
    path = str(tmp_path / "frame.bin")
    with open(path, "wb") as f:
        f.write(np.uint64(len(cl)).tobytes())
        f.write(cl.tobytes())
    r = subprocess.run([exe, path], capture_output=True, text=True, env={**os.environ, "ASAN_OPTIONS": "detect_leaks=1"})
    assert r.returncode == 0, r.stderr[-3000:]
    assert "ERROR" not in r.stderr and "runtime error" not in r.stderr, r.stderr[-3000:]
    words = r.stdout.split()
    got = {words[i]: int(words[i + 1]) for i in range(0, len(words), 2)}
    assert got["tracks"] > 300 and got["links"] > 10 and got["fits"] > 300
