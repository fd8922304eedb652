"""Host logic of bench.py's roofline bookkeeping (no GPU): which side of the roofline a set of sampled launches is
reported against, and that merged families add up.  DESIGN.md section 9 "Which side of the roofline"."""
import numpy as np

import bench

TP = {"f64_contract": 28.2, "tf32x3_contract": 234.7, "f64_issue": 37.2, "src": "test"}
HBM = 6543.1


def _prof(ms, live, n, r, launches):
    fl = [2.0 * n * r * lv * nl for lv, nl in zip(live, launches)]
    return {"ms": np.array(ms, dtype=float), "flops": np.array(fl), "launches": np.array(launches)}


def test_narrow_batch_on_a_large_u_is_reported_on_the_hbm_side():
    n = r = 20000
    # 14 live columns, 0.6 ms per tcgen05 launch: 3.2 GB of U pairs per launch -> HBM-bound by any model
    prof = _prof([8.8, 8.8, 6.0, 6.0], [14, 14, 14, 14], n, r, [10, 10, 10, 10])
    fams = bench.family_rooflines(prof, TP, {}, None, geom=(n, r, 1), hbm_peak=HBM)
    assert [f["binding"] for f in fams] == ["hbm"] * 4
    d = bench.binding_side(fams[2])
    by = n * r * 8.0 + 14 * (n + r) * 8.0
    assert d["bound"] == "hbm" and d["unit"] == "GB/s" and d["peak"] == HBM
    assert abs(d["achieved"] - by / 0.6e-3 / 1e9) < 1e-6 * d["achieved"]
    assert abs(d["frac"] - d["achieved"] / HBM) < 1e-12
    assert d["tensor_side"]["unit"] == "TFLOP/s" and d["tensor_side"]["peak"] == TP["tf32x3_contract"]


def test_wide_batch_and_l2_resident_operands_stay_on_the_tensor_side():
    # 900 live columns at n = 20000: 58 flop per byte for the FP64 kernel, far above its ridge point of 4.3
    prof = _prof([22.0, 22.0, 3.4, 3.4], [900] * 4, 20000, 20000, [1, 1, 1, 1])
    fams = bench.family_rooflines(prof, TP, {}, None, geom=(20000, 20000, 1), hbm_peak=HBM)
    assert fams[0]["binding"] == "tensor" and fams[2]["binding"] == "tensor"
    d = bench.binding_side(fams[0])
    assert d["bound"] == "tensor" and "hbm_side" in d and "hbm" not in d
    # a single n = 2000 bandwidth (32 MB of U) fits L2: tensor side whatever the width
    prof = _prof([0.03, 0.03, 0.02, 0.02], [8] * 4, 2000, 2000, [1, 1, 1, 1])
    fams = bench.family_rooflines(prof, TP, {}, None, geom=(2000, 2000, 1), hbm_peak=HBM)
    assert all(f["binding"] == "tensor" for f in fams)


def test_single_tf32_mode_counts_four_byte_operands_and_the_full_tf32_peak():
    n = r = 20000
    prof = _prof([0.0, 0.0, 4.0, 4.0], [0, 0, 15, 15], n, r, [0, 0, 10, 10])
    three = bench.family_rooflines(prof, TP, {}, None, geom=(n, r, 1), hbm_peak=HBM)
    one = bench.family_rooflines(prof, TP, {}, None, geom=(n, r, 1), hbm_peak=HBM, single_tf32=True)
    assert len(three) == len(one) == 2
    assert one[0]["peak"] == 3.0 * three[0]["peak"] and "1xTF32" in one[0]["kernel"]
    ub3 = three[0]["hbm"]["algorithmic_bytes_per_launch"] - 15 * (n + r) * 8.0
    ub1 = one[0]["hbm"]["algorithmic_bytes_per_launch"] - 15 * (n + r) * 8.0
    assert abs(ub3 - n * r * 8.0) < 1.0 and abs(ub1 - n * r * 4.0) < 1.0


def test_merged_families_add_up():
    n = r = 2000
    prof = _prof([30.0, 29.0, 4.7, 4.7], [60, 60, 357, 357], n, r, [220, 220, 91, 91])
    fams = bench.family_rooflines(prof, TP, {}, None, geom=(n, r, 5), hbm_peak=HBM)
    m = bench.merge_families(fams, (2, 3))
    assert m["sampled_launches"] == 182 and abs(m["sampled_ms"] - 9.4) < 1e-12
    fl = sum(f["avg_flops_per_launch"] * f["sampled_launches"] for f in fams[2:])
    assert abs(m["achieved"] - fl / 1e12 / 9.4e-3) < 1e-9 * m["achieved"]
    by = sum(f["hbm"]["algorithmic_bytes_per_launch"] * f["sampled_launches"] for f in fams[2:])
    assert abs(m["hbm"]["achieved"] - by / 9.4e-3 / 1e9) < 1e-9 * m["hbm"]["achieved"]
    # five bandwidths of n = 2000 are 160 MB of U per launch (> L2) at 17 flop per byte: the HBM side binds
    assert m["binding"] == "hbm"
    tw = bench.time_weighted({"ms": prof["ms"], "flops": prof["flops"], "launches": prof["launches"]}, TP)
    assert set(tw) == {"fp64_dmma", "tcgen05_3xtf32", "note"}
    assert abs(tw["tcgen05_3xtf32"]["frac"] - tw["tcgen05_3xtf32"]["achieved"] / TP["tf32x3_contract"]) < 1e-12


def test_traffic_table_is_read_from_the_committed_csv():
    t = bench.traffic_table()
    assert {"config1_dmma_full_width", "config1_tcgen05_full_width"} <= set(t)
    for key, (nbytes, source) in t.items():
        assert nbytes > 0 and source.startswith("profiles/")
