"""bench.py's stdout line, built from fake numbers through the same code path main() uses
(rooflines -> workload_scalars -> assemble_line -> emit): it must stay one compact JSON object the
driver can parse -- round 2's line grew to 22 KB and was recorded as unmeasured."""
import json

import bench


def _fake_measurement(w, steps):
    kinds = {"fwd_stats": (30.0 * steps, steps), "recompute_ds": (31.0 * steps, 2 * steps),
             "dh": (29.123456789 * steps, 2 * steps), "dw": (33.3 * steps, 2 * steps)}
    peaks = bench.load_peaks()
    roofs = bench.rooflines(w, 8192, steps, kinds, 130.0 * steps, peaks)
    return roofs, peaks


def test_default_line_is_compact_and_complete():
    w = bench.I.CONFIGS[bench.WORKLOADS[bench.HEADLINE]]
    steps = 20
    roofs, _ = _fake_measurement(w, steps)
    assert len(roofs) == 4
    others = {}
    for name in ("cfg1", "cfg2", "cfg3"):
        wo = bench.I.CONFIGS[bench.WORKLOADS[name]]
        r, _ = _fake_measurement(wo, 4)
        m = {"ms_per_step": 80.123456789, "value": 305662.123456, "step_tflops": 1284.6123,
             "rooflines": r, "e2e": {"ms_per_step": 81.98765432} if name != "cfg3" else None}
        others[name] = bench.workload_scalars(m)
        assert others[name]["worst_kind"] == "dw"          # the slowest per flop of the fakes
    clocks = {"sm_mhz": 1230.0, "sm_max_mhz": 1965.0, "power_w_max": 1001.8, "samples": 60,
              "reasons": ["sw_power_cap"], "per_gpu": [{"index": 0, "sm_mhz": 1230.0}]}
    e2e = {"value": 75000.123, "unit": "scored tokens/s", "ms_per_step": 109.8,
           "h2d_bytes_per_step": 134_300_000, "d2h_bytes_per_step": 134_217_748,
           "pass": "x" * 300, "loss": 0.1}
    cpu = {"value": 3.21, "unit": "scored tokens/s", "cores": 16, "kind": "oracle",
           "sample": "1 x 64 tokens of cfg4_large_vocab (full D=8192, V=256000), fwd+bwd, 12.3 s, fp64 numpy",
           "seconds": 12.3, "one_thread": {"value": 0.4, "cores": 1, "sample": "y" * 100},
           "config0_full": {"value": 1.0}}
    out = bench.assemble_line(w, value=76543.21, ms_per_step=107.0, T=8192, world=1, steps=steps,
                              warmup=5, exchange="none", clocks=clocks, gpu_launches=17 * steps,
                              roofs=roofs, step_ms=107.0, e2e=e2e, cpu=cpu, workloads=others)
    line = bench.emit(out)
    assert len(line) < 4096 and "\n" not in line
    d = json.loads(line)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step",
              "higher_is_better", "scaling", "vs_baseline", "dtype", "data", "config", "clocks",
              "gpu_launches", "roofline", "e2e", "cpu_baseline", "workloads"):
        assert k in d, k
    assert d["config"]["workload"] == w.name and "model" not in d["config"]
    assert d["value"] > 0 and d["gpu_launches"] > 0 and d["n_gpus"] == 1
    rf = d["roofline"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic", "kernel", "launch_ms",
              "flops_per_launch", "frac_of_burst", "frac_of_sustained"):
        assert k in rf, k
    assert rf["bound"] == "tensor" and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-12
    assert rf["kind"] == "dw"                               # the kind with the most time per step
    for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert k in d["e2e"]
    assert "pass" not in d["e2e"]
    for k in ("value", "unit", "cores", "kind", "sample"):
        assert k in d["cpu_baseline"]
    assert d["cpu_baseline"]["one_thread"]["value"] == 0.4
    # nothing nested below the per-workload scalars, no list of roofline objects anywhere
    assert "rooflines" not in d
    for name, sc in d["workloads"].items():
        assert all(not isinstance(v, (dict, list)) for v in sc.values()), name


def test_emit_refuses_an_oversized_line():
    import pytest
    with pytest.raises(AssertionError):
        bench.emit({"x": "y" * 5000})
