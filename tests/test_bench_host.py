"""Host-side logic of bench.py that needs no GPU: byte/flop models, roofline selection, workload description."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import arche_inputs as ai  # noqa: E402
import bench  # noqa: E402


def test_bytes_per_point_models():
    fused = bench.bytes_per_point(64, True)
    h = 16.0 * 40 / 64                       # nx/2+1 = 33 stored columns padded to 40
    assert fused["fft_y"] == 2 * h and fused["fft_inv_z_potential"] == 5 * h and fused["density"] == 24 + h
    streamed = bench.bytes_per_point(384, False)
    h = 16.0 * 200 / 384
    assert abs(streamed["potential_g"] - 5 * h) < 1e-12 and streamed["vi_r"] == 40 and streamed["density_r"] == 24
    assert "density" not in streamed and "potential_g" not in fused
    assert abs(streamed["stress_fields"] - (3 * h + 8)) < 1e-12       # f1: once per stress call, not per iteration
    # one SCF iteration of the streamed form moves 18 h + 80 (+ 8 per mu evaluation) bytes per point
    per_iter = sum(streamed[k] * (2 if k == "fft_y" else 1) for k in streamed
                   if k not in ("mix", "mu_pass", "stress_fields"))
    assert abs(per_iter - (18 * h + 80)) < 1e-9


def test_roofline_entry_picks_the_binding_bound():
    bpp = bench.bytes_per_point(384, False)
    ng = 384 ** 3
    args = (6547.2, "measured", 36.84, "measured fp64")
    e = bench.roofline_entry("potential_g", 0.357, ng, bpp, *args)
    assert e["bound"] == "hbm" and 0.95 < e["frac"] < 1.05
    e = bench.roofline_entry("density_r", 0.720, ng, bpp, *args)
    assert e["bound"] == "alu" and 0.35 < e["frac"] < 0.5 and e["unit"] == "TFLOP/s" and e["peak"] == 36.84
    # the plain c2r pass of the streamed form carries no epilogue arithmetic: HBM bound only
    e = bench.roofline_entry("fft_inv_x_vi", 0.244, ng, bpp, *args)
    assert e["bound"] == "hbm"
    # ion-grid sums: flops per (ion, stored half-spectrum point) pair against the fp64 peak
    pairs = 2000.0 * 200 * 384 * 384
    e = bench.roofline_entry("force", 48.8, ng, bpp, *args, pairs=pairs)
    assert e["bound"] == "alu" and abs(e["achieved"] - 16 * pairs / 48.8e-3 / 1e12) < 1e-9 and 0.45 < e["frac"] < 0.6
    assert abs(bench.FP64_DERIVED_TFLOPS - 37.22) < 0.01


def test_ncu_traffic_is_parsed_from_the_committed_capture(tmp_path, monkeypatch):
    p = tmp_path / "cap.csv"
    p.write_text("class,kernel,time_us,dram_bytes_read,dram_bytes_write\n"
                 "potential_g,pointwise_g_kernel<LoadPotentialG>,363.0,1420000000,890000000\n"
                 "potential_g,pointwise_g_kernel<LoadPotentialG>,361.0,1440000000,890000000\n"
                 ",unclassified_kernel,1.0,5,5\n")
    monkeypatch.setattr(bench, "NCU_TRAFFIC_CSV", str(p))
    t = bench.ncu_traffic()
    assert list(t) == ["potential_g"] and abs(t["potential_g"] - 2.32e9) < 1
    monkeypatch.setattr(bench, "NCU_TRAFFIC_CSV", str(tmp_path / "missing.csv"))
    assert bench.ncu_traffic() == {}                      # absent capture: traffic stays null, nothing is invented


def test_settings_per_workload_and_default_is_the_largest_config():
    assert bench.tol_for("c2")["mix_w_fixed"] == 0.95 and "mix_mu_tol" not in bench.tol_for("c2")
    t4 = bench.tol_for("c4")
    assert t4["mix_w_fixed"] == 0.0 and t4["mix_mu_tol"] == 1e-3 and t4["scf_tol_F"] == 1e-10
    cfg = ai.make_config("c5")
    w = bench.workload_config(cfg, "c5")
    assert "[384, 384, 384]" in w["workload"] and "56.62 M points" in w["workload"] and "exceed the 126 MB L2" in w["l2"]
    assert "P:311" in bench.workload_config(ai.make_config("c4"), "c4")["mixing"]


def test_workload_description_and_configs():
    for name, ions, grid in (("c1", 16, 32), ("c2", 128, 64), ("c3", 256, 128), ("c4", 1024, 192)):
        cfg = ai.make_config(name)
        assert len(cfg["Z"]) == ions and int(cfg["grid"][0]) == grid
        w = bench.workload_config(cfg, name)
        assert name in w["workload"] and "stop_rule" in w
    cfg = ai.make_config("c5", grid=96)
    assert len(cfg["Z"]) == 2000 and int(cfg["grid"][2]) == 96
