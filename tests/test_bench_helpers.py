"""CPU-side checks of bench.py's accounting: the algorithmic bytes are SURVEY.md 8(d)'s table, both arms carry the
same `config`, and the parity key separates flipped groups from the others."""
import argparse
import importlib.util
import os

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
spec = importlib.util.spec_from_file_location("bench", os.path.join(ROOT, "bench.py"))
bench = importlib.util.module_from_spec(spec)
spec.loader.exec_module(bench)


def test_build_bytes_are_the_survey_table():
    # 256^3: (n - 1)/7 nodes, 3 sort passes: 36 + (8 + 72) + 84 + (8 + 24/7) + (32 + 72/7) = 253.71 B/cell
    n = 256 ** 3
    nn = (n - 1) // 7
    assert abs(bench.build_bytes_per_cell(n, nn, 3) - (36 + 80 + 84 + 8 + 32 + 96 * nn / n)) < 1e-9
    assert abs(bench.build_bytes_per_cell(n, nn, 3) - 253.714) < 1e-3
    assert bench.build_bytes_per_cell(n, nn, 0) == bench.build_bytes_per_cell(n, nn, 3) - 80      # all keys equal: no sort
    assert bench.IMPL_EXTRA_BYTES_PER_CELL == 9.0


def test_both_arms_share_one_config_object():
    class W:
        name, n, theta, G = "turb256", 16777216, 0.5, 1.0
    a, b = bench.make_config(W, 1), bench.make_config(W, 1)
    assert a == b and a["workload"] == "turb256" and "l2" in a and "parallelism" in a


def test_parity_key_counts_flips_and_keeps_them_apart():
    class W:
        n = 32 * 6
    rng = np.random.default_rng(1)
    perm = rng.permutation(W.n).astype(np.int64)
    phi_orc = -rng.uniform(1.0, 2.0, W.n)
    phi_gpu = phi_orc * (1 + 1e-8)
    cnt = np.tile(np.array([10, 20, 5]), (6, 1))
    c64 = [cnt[0:3].copy(), cnt[3:6].copy()]
    c64[1][1, 0] += 1                                   # group 4 flipped: one node accepted instead of opened
    phi_gpu[perm[32 * 4:32 * 5]] *= 1 + 3e-5             # ... and its Phi differs at the tree code's level
    sample = {"runs": [(0, 3), (3, 6)], "counts": c64, "perm": perm}
    ev = cnt[:, 0] + cnt[:, 1]
    out = bench.parity_key(W, phi_gpu, cnt, ev, phi_orc, sample)
    assert out["groups"] == 6 and out["flips_fp32_vs_fp64"] == 1 and out["targets"] == W.n
    assert out["max_rel"] < 2e-8 and 2e-5 < out["max_rel_flipped_groups"] < 4e-5 and out["pass"]
    ev2 = ev.copy(); ev2[2] += 1                        # the Phi kernel lost or doubled an entry
    assert not bench.parity_key(W, phi_gpu, cnt, ev2, phi_orc, sample)["pass"]
