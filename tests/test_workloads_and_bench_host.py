"""CPU checks of host-side pieces that carry no arithmetic of the method: the pair-creation-order stand-in of
workloads.py (DESIGN.md section 4 / 5) and bench.py's recorded-traffic bookkeeping (a figure captured on other kernel
sources must be reported as stale, never as a number)."""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2110_09214_b200 import workloads as W  # noqa: E402


def test_pair_creation_order_is_a_seeded_permutation_that_interleaves_the_signs():
    base = W.make_workload(1)
    wl = W.pair_creation_order(base)
    perm = wl.meta["perm"]
    assert sorted(perm.tolist()) == list(range(base.n_charges))
    assert np.array_equal(wl.xyzq, base.xyzq[perm])
    assert wl.verts is base.verts and wl.sigma is base.sigma and wl.eps_pp == base.eps_pp
    # the generator stores all electrons, then all ions; the stand-in interleaves them: many sign changes
    assert (np.diff(np.sign(base.xyzq[:, 3])) != 0).sum() == 1
    assert (np.diff(np.sign(wl.xyzq[:, 3])) != 0).sum() > base.n_charges // 4
    again = W.pair_creation_order(W.make_workload(1))
    assert np.array_equal(again.xyzq, wl.xyzq)                     # seeded: the same order every time
    other = W.pair_creation_order(base, seed=1)
    assert not np.array_equal(other.xyzq, wl.xyzq)
    assert W.pair_creation_order(W.make_workload(5, mesh_div=8, point_div=64)).n_charges == 0   # no charges: unchanged


def test_recorded_traffic_is_null_when_the_kernel_sources_changed(tmp_path, monkeypatch):
    import bench
    h = bench.kernel_source_hash()
    assert len(h) == 16 and h == bench.kernel_source_hash()
    rec = {"kernel_source_hash": h, "configs": {"3": {"bytes_per_evaluation": 123, "capture": "x"}}}
    prof = tmp_path / "profiles"
    prof.mkdir()
    (prof / "r02_traffic.json").write_text(json.dumps(rec))
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    monkeypatch.setattr(bench, "kernel_source_hash", lambda: h)
    val, src = bench.recorded_traffic(3)
    assert val == 123 and "recorded" in src
    val, src = bench.recorded_traffic(4)
    assert val is None and "no capture" in src
    monkeypatch.setattr(bench, "kernel_source_hash", lambda: "0" * 16)
    val, src = bench.recorded_traffic(3)
    assert val is None and src.startswith("stale")
    (prof / "r02_traffic.json").unlink()
    val, src = bench.recorded_traffic(3)
    assert val is None and src.startswith("no record")
