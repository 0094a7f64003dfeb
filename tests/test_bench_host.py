"""Host logic of bench.py that needs no GPU: the ncu-counter summary that feeds the roofline (`--ncu-summary`) and the
roofline arithmetic itself (achieved = measured thread-instructions per step x steps per launch / launch duration)."""
import csv
import importlib
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench():
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    return importlib.import_module("bench")


def _fake_ncu_csv(path):
    hdr = ["ID", "Process ID", "Process Name", "Host Name", "Kernel Name", "Context", "Stream", "Block Size", "Grid Size", "Device", "CC",
           "Section Name", "Metric Name", "Metric Unit", "Metric Value"]
    rows = []
    kid = 0
    for name, n_launch, tinst, winst in (("void vpk::beam_kernel<(int)0, (int)7>(vpk::Ctx, vpk::SourceBuf)", 2, 4000.0, 160.0),
                                         ("void vpk::beam_kernel<(int)1, (int)7>(vpk::Ctx, vpk::SourceBuf)", 2, 1000.0, 40.0),
                                         ("void vpk::voxel_kernel<(int)0, (bool)0, (int)7>(vpk::Ctx, vpk::Queue)", 4, 3000.0, 100.0)):
        for _ in range(n_launch):
            for m, v in (("gpu__time_duration.sum", "1,000"), ("smsp__thread_inst_executed.sum", "%.0f" % tinst), ("smsp__inst_executed.sum", "%.0f" % winst),
                         ("dram__bytes_read.sum", "30"), ("dram__bytes_write.sum", "10"), ("lts__t_bytes.sum", "800"), ("lts__t_sectors_op_red.sum", "12"),
                         ("lts__t_sector_hit_rate.pct", "50")):
                rows.append([str(kid), "1", "python", "h", name, "1", "7", "(256, 1, 1)", "(1, 1, 1)", "0", "10.0", "s", m, "u", v])
            kid += 1
    with open(path, "w", newline="") as f:
        f.write("==PROF== Connected\n")
        w = csv.writer(f, quoting=csv.QUOTE_ALL)
        w.writerow(hdr)
        w.writerows(rows)


def test_ncu_summary_divides_the_counters_by_the_counted_steps(tmp_path, monkeypatch):
    b = _bench()
    ncu = tmp_path / "m.csv"
    _fake_ncu_csv(ncu)
    log = tmp_path / "bench.log"
    log.write_text("noise\n" + json.dumps({"profile_units": {"steps_run": 2, "ct_steps_per_step": 6, "slab_steps_per_step": 5}}) + "\n")
    out = tmp_path / "inst.csv"
    monkeypatch.setattr(b, "INST_CSV", str(out))
    b.ncu_summary(str(ncu), str(log), "cfgA")
    b.ncu_summary(str(ncu), str(log), "cfgB")                 # a second config is appended, the first kept
    rows = {(r["config"], r["kernel"]): r for r in csv.DictReader(open(out))}
    assert set(rows) == {("cfgA", "beam_kernel"), ("cfgA", "voxel_kernel"), ("cfgB", "beam_kernel"), ("cfgB", "voxel_kernel")}
    r = rows[("cfgA", "beam_kernel")]                          # both stages: 2 x 4000 + 2 x 1000 thread instructions over 2 x 5 slab steps
    assert int(r["launches"]) == 4 and int(r["units"]) == 10 and abs(float(r["thread_inst_per_unit"]) - 1000.0) < 1e-9
    assert abs(float(r["lanes_per_inst"]) - 25.0) < 1e-9 and abs(float(r["dram_bytes_per_unit"]) - 16.0) < 1e-9
    v = rows[("cfgA", "voxel_kernel")]                         # 4 x 3000 over 2 x 6 voxel steps
    assert int(v["units"]) == 12 and abs(float(v["thread_inst_per_unit"]) - 1000.0) < 1e-9 and abs(float(v["red_sectors_per_unit"]) - 4.0) < 1e-9
    assert abs(float(v["l2_hit_pct"]) - 50.0) < 1e-9
    assert b.load_inst_counts("cfgA")["voxel_kernel"]["units"] == "12" and b.load_inst_counts("none") is None


def test_roofline_arithmetic(tmp_path, monkeypatch):
    b = _bench()
    out = tmp_path / "inst.csv"
    with open(out, "w") as f:
        f.write("config,kernel,launches,time_ms,units,thread_inst_per_unit,warp_inst_per_unit,lanes_per_inst,dram_bytes_per_unit,l2_bytes_per_unit,red_sectors_per_unit,l2_hit_pct\n")
        f.write("cfg,beam_kernel,1,1,1,400.0,14,28.5,3.0,12.0,0.0,40.0\ncfg,voxel_kernel,1,1,1,500.0,18,27.0,1.0,70.0,1.5,75.0\n")
    monkeypatch.setattr(b, "INST_CSV", str(out))
    rec = {"steps": 2, "ms_per_step": 10.0, "slab_steps_per_step": 4.0e9, "ct_steps_per_step": 2.0e9,
           "timing_ms_per_step": {"beamline": 6.0, "voxel": 3.0}, "launches_per_step": {"beamline": 12.0, "voxel": 6.0}, "red_ceiling": (2.0e11, 1)}
    kr = {r["kernel"]: r for r in b.rooflines(rec, "cfg", 6000.0, 2000.0, "measured")}
    peak = 148 * 4 * 32 * 2000.0e6 / 1e9
    bk = kr["beam_kernel"]
    assert abs(bk["peak"] - peak) < 1e-6 and abs(bk["avg_launch_ms"] - 0.5) < 1e-12 and abs(bk["units_per_launch"] - 4.0e9 / 12) < 1
    assert abs(bk["achieved"] - 400.0 * 4.0e9 / 6.0e-3 / 1e9) < 1e-3 and abs(bk["frac"] - bk["achieved"] / peak) < 1e-12
    assert abs(bk["frac_survey_count"] - b.SURVEY_INST_PER_STEP * 4.0e9 / 6.0e-3 / 1e9 / peak) < 1e-12 and abs(bk["share_of_step"] - 0.6) < 1e-12
    vk = kr["voxel_kernel"]
    assert abs(vk["hbm"]["achieved"] - 10.0 * 2.0e9 / 3.0e-3 / 1e9) < 1e-6 and abs(vk["hbm"]["frac"] - vk["hbm"]["achieved"] / 6000.0) < 1e-12
    assert abs(vk["red"]["achieved_ops_per_s"] - 2.0e9 / 3.0e-3) < 1 and abs(vk["red"]["frac"] - vk["red"]["achieved_ops_per_s"] / 2.0e11) < 1e-12
    assert abs(vk["traffic"] - 1.0 * 2.0e9 / 6) < 1 and abs(vk["l2"]["achieved_GBps"] - 70.0 * (2.0e9 / 6) / 0.5e-3 / 1e9) < 1e-6
    # a config without committed counters still reports the survey-count fraction, and says so
    none = b.rooflines(rec, "other", 6000.0, 2000.0, "measured")[0]
    assert none["frac"] is None and none["frac_survey_count"] > 0 and "no committed" in none["inst_source"]
