"""Host logic of bench.py's output: the last stdout line must stay small enough for the driver to parse (round 2's
31.9 KB line was cut off and nothing was recorded), and the `l2` statement must follow the predicate that switches the
L2 flush.  No GPU needed: the line is built from canned numbers."""
import json

import bench


def _canned_line(note_len=600):
    long = "x" * note_len
    roof = {"bound": "alu", "achieved": 14.7312345678, "peak": 18.6112345678, "unit": "T FP64 instr/s", "frac": 0.7915123456,
            "peak_source": "derived: 148 SM x 64 FP64 lanes x sm_max_mhz (DESIGN.md 6)", "algorithmic_fp64_instr_per_launch": 6.05e12,
            "tflops": 26.8, "peak_tflops": 37.22, "flop_frac": 0.72, "frac_at_held_clock": 0.79, "frac_of_measured_issue_rate": 0.8,
            "flop_frac_of_measured_dfma": 0.82, "flop_frac_ordered_convention": 1.15, "note": long, "kernel": "pair_force_band_kernel",
            "kernel_avg_ms": 410.5, "kernel_launches_timed": 9, "kernel_launches_per_force_evaluation": 1.0,
            "kernel_share_of_step": 0.9988, "traffic": 1.5e9, "traffic_source": "profiles/r02_traffic.csv", "traffic_what": long,
            "algorithmic_dram_bytes_per_force_evaluation": 33.5e6, "traffic_ratio": 44.8, "workspace_bytes": 673000000}
    return {
        "metric": "pair-interactions/s", "value": 2.674e12, "unit": "pair-interactions/s", "n_gpus": 1, "steps": 20, "warmup": 5,
        "ms_per_step": 1233.8, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "grav2d_1m", "model": "grav2d", "N": 1048576, "eps": 1e-3, "dt": 0.005, "step": long,
                   "parallelism": "1 GPU", "l2": "L2 flushed (256 MiB write) before every timed step"},
        "options": {"pair_ctas": 296, "pair_variant": 1, "pair_slots": 1, "graph": -1, "hmf_grid": 0, "hmf_variant": 0,
                    "pair_precision": 0, "pair_symmetric": 2},
        "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": ["sw_power_cap"], "samples": 1200},
        "e2e": {"value": 2.67e12, "unit": "pair-interactions/s", "h2d_bytes_per_step": 16777216.0, "d2h_bytes_per_step": 16777216.0,
                "steps_per_call": 2, "note": long},
        "gpu_launches": 180, "roofline": roof, "energy": {"ms_per_call": 400.0, "what": long, "pair_interactions_per_s": 2.7e12},
        "cpu_baseline": {"value": 3.4e9, "unit": "pair-interactions/s", "cores": 16, "kind": "oracle", "sample": long, "note": long},
        "others": {"k%d" % i: {"roofline": roof, "note": long} for i in range(16)},
        "others_file": "gpurun_out/bench_others.json",
    }


def test_headline_is_small_and_complete():
    line = _canned_line()
    assert len(json.dumps(line)) > 30000                 # the shape that broke round 2
    h = bench.headline(line)
    text = json.dumps(h)
    assert len(text) < 4096 and len(text) <= bench.HEADLINE_MAX_BYTES
    assert "\n" not in text and "others" not in h
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in h, k
    assert h["config"]["workload"] == "grav2d_1m" and "step" not in h["config"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in h["roofline"], k
    assert abs(h["roofline"]["frac"] - h["roofline"]["achieved"] / h["roofline"]["peak"]) < 1e-4
    assert set(h["e2e"]) == {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "steps_per_call"}
    assert set(h["cpu_baseline"]) == {"value", "unit", "cores", "kind", "sample"}
    assert h["value"] == 2.674e12 and h["vs_baseline"] is None


def test_headline_keeps_the_contract_keys_when_strings_are_huge():
    h = bench.headline(_canned_line(note_len=20000))
    assert len(json.dumps(h)) <= bench.HEADLINE_MAX_BYTES
    assert {"value", "roofline", "e2e", "cpu_baseline", "clocks", "config"} <= set(h)
    assert h["roofline"]["traffic"] == 1.5e9


def test_headline_keeps_a_null_traffic():
    line = _canned_line()
    line["roofline"]["traffic"] = None
    assert bench.headline(line)["roofline"]["traffic"] is None


def test_reference_line_passes_through():
    ref = {"impl": "reference", "metric": "pair-interactions/s", "value": 3.4e9, "unit": "pair-interactions/s", "n_gpus": 1,
           "steps": 3, "warmup": 1, "ms_per_step": None, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "config": {"workload": "grav2d_1m"},
           "cpu_baseline": {"value": 3.4e9, "unit": "u", "cores": 16, "kind": "oracle", "sample": "s"},
           "e2e": {"value": 3.4e9, "unit": "u", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    h = bench.headline(ref)
    assert h["impl"] == "reference" and h["e2e"]["h2d_bytes_per_step"] == 0 and h["gpu_launches"] == 0


def test_l2_statement_follows_the_flush_predicate(inputs):
    ws = dict(inputs.WORKLOADS, **inputs.TABLE1_WORKLOADS)
    w = ws["hmf_1e6"]                                     # 16 MB state: fits L2; the default kernel keeps it on chip
    assert bench.l2_statement(w, hmf_resident=True).startswith("not flushed")
    assert bench.l2_statement(w, hmf_resident=False).startswith("L2 flushed")      # fallback to the streaming kernels
    assert bench.l2_statement(w) == bench.l2_statement(w, hmf_resident=True)        # what the reference arm prints
    assert bench.l2_statement(ws["hmf_5e7"], hmf_resident=False).startswith("inputs larger than L2")
    assert bench.l2_statement(ws["ring_16k"]).startswith("L2 flushed")
    assert bench.workload_config(w, 1, l2="abc")["l2"] == "abc"
