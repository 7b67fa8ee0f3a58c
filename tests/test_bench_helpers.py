"""Host-side helpers of bench.py that need no GPU: the ncu figures it quotes are read from the
summaries committed under profiles/, so a renamed file or a changed line format must fail here and
not silently turn `roofline.traffic` into null."""
import importlib.util
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def load_bench():
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_ncu_figures_are_found_in_profiles():
    bench = load_bench()
    import re
    for kernel in ("tiled_triplet_kernel", "neighbour_cell_kernel"):
        path = os.path.join(ROOT, "profiles", bench.TRAFFIC_PROFILES[kernel])
        fpl = int(re.search(r"frames_per_launch=(\d+)", open(path).read()).group(1))
        assert fpl == 117                                  # config 4's default batch: what bench.py runs
        traffic, src = bench.ncu_traffic(kernel, fpl)
        assert src and os.path.exists(os.path.join(ROOT, src))
        assert traffic and 1e8 < traffic < 1e11            # bytes per launch
        assert bench.ncu_traffic(kernel, fpl - 1)[0] is None    # another batch size: not quoted
        busy = bench.ncu_lsu_busy(kernel)
        assert busy and 0.3 < busy <= 1.0


def test_profiles_hold_text_only_and_name_their_command():
    pdir = os.path.join(ROOT, "profiles")
    for fn in os.listdir(pdir):
        assert fn.endswith((".md", ".txt", ".csv")), fn
        if fn.endswith(".md"):
            text = open(os.path.join(pdir, fn)).read()
            assert "ncu " in text and "bench.py" in text, fn


def test_metric_and_workload_follow_baseline_json():
    import json
    bench = load_bench()
    base = json.load(open(os.path.join(ROOT, "BASELINE.json")))
    assert "triplets" in base["metric"] and bench.UNIT == "triplets/s"
    w = bench.WORKLOADS[bench.WORKLOAD_INDEX]
    assert (w.n, w.n_frames, w.n_r, w.n_t) == (32768, 500, 64, 64) and abs(w.r_max - 0.7) < 1e-12
