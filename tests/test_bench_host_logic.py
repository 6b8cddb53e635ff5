"""Host-side logic of bench.py (no GPU): the sampling plan of the CPU-baseline / reference legs carries the SURVEY.md 8(d)
budget labels, the stored ncu traffic figure is dropped when the kernel sources change, and the config dictionary is the
same object for both arms."""
import importlib
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
bench = importlib.import_module("bench")
from paper_2208_06559_b200 import workloads as W  # noqa: E402


def test_oracle_plan_labels_follow_the_survey_budget():
    plans = {n: bench._oracle_plan(w) for n, w in W.CONFIGS.items()}
    assert [plans[n]["label"] for n in ("c1", "c2", "c3", "c4", "c5")] == ["measured", "measured", "measured", "scaled", "extrapolated"]
    assert plans["c1"]["chains"] == 1 and plans["c1"]["threads"] == 1           # one chain keeps one thread busy
    assert plans["c2"]["n_rods"] == 100 and plans["c3"]["n_rods"] == 500        # real chains of the workload
    assert plans["c4"]["chains"] == 1 and plans["c4"]["n_rods"] == 2000          # one chain x one step, x C stated as scaled
    assert plans["c5"]["n_rods"] == 1000 and abs(plans["c5"]["scale"] - (30003 / 3003) ** 3) < 1e-9
    for n, w in W.CONFIGS.items():
        text = bench._oracle_sample_text(w, plans[n], 3, 1.5)
        assert text.startswith(plans[n]["label"])


def test_traffic_is_dropped_when_kernel_sources_change(tmp_path, monkeypatch):
    sha = bench._sources_sha16()
    prof = tmp_path / "profiles"
    prof.mkdir()
    (prof / "traffic.json").write_text(json.dumps({"c5": {"bytes": 123, "commit": "abc", "file": "f.csv", "sources_sha16": sha},
                                                   "c4": {"bytes": 5, "commit": "old", "file": "g.csv", "sources_sha16": "0" * 16}}))
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    monkeypatch.setattr(bench, "_sources_sha16", lambda: sha)
    assert bench._traffic("c5")[0] == 123 and "abc" in bench._traffic("c5")[1]
    val, why = bench._traffic("c4")
    assert val is None and "stale" in why
    assert bench._traffic("c3")[0] is None


def test_committed_traffic_stamp_matches_the_tree():
    """the ncu figures in profiles/traffic.json were captured with the kernels of this tree."""
    t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    for name in ("c2", "c3", "c4", "c5"):
        assert t[name]["sources_sha16"] == bench._sources_sha16(), name
        assert os.path.exists(os.path.join(ROOT, t[name]["file"]))


def test_config_dictionary_is_shared_by_both_arms():
    w = W.CONFIGS["c5"]
    a = bench._config(w, w.n_chains, bench._l2_text(w, False, 7206 * 10 ** 6))
    assert list(a) == ["workload", "n_chains_per_gpu", "n_rods", "M", "dt", "hstar", "flow", "Wi", "l2"]
    assert a["workload"] == "c5" and a["M"] == 30003
