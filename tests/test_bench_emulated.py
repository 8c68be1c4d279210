"""bench.py's product arm, executed end to end on a box without a GPU: run_ours / run_sweep / run_fill_floor / run_wave at
tiny sizes against the emulated library (tests/native/libchemora_emu.cpp) with the few torch.cuda calls bench.py makes
(events, streams, pinned memory) shimmed.  No number printed here means anything; what is checked is that the script
runs through every branch it takes on the GPU box -- runtime sweep, timed steps with per-kernel timing, the two-handle
end-to-end pipeline, the FP64 probe, the CPU baseline -- and prints ONE JSON line with the keys of the bench contract
(metric byte-identical to BASELINE.json, roofline, cpu_baseline, e2e, gpu_launches, clocks).  bench.py was edited
without GPU access in round 2; a NameError in its line assembly would cost the round's headline measurement."""
import contextlib
import importlib.util
import json
import os
import time
import types

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture
def bench(monkeypatch):
    import torch
    from paper_1307_6488_b200 import binding
    from tests.conftest import build_emulator
    monkeypatch.setattr(binding, "LIB_PATH", build_emulator("libchemora_emu", shared=True))
    monkeypatch.setattr(binding, "_lib", None)
    avail = {"v": True}                               # bench.py must see a device, the binding must use host memory
    monkeypatch.setattr(torch.cuda, "is_available", lambda: avail["v"])
    monkeypatch.setattr(torch.cuda, "set_device", lambda d: None)
    monkeypatch.setattr(torch.cuda, "synchronize", lambda *a, **k: None)

    class Event:
        def __init__(self, enable_timing=False):
            self.t = None

        def record(self):
            self.t = time.perf_counter()

        def elapsed_time(self, other):
            return (other.t - self.t) * 1e3

    monkeypatch.setattr(torch.cuda, "Event", Event)
    monkeypatch.setattr(torch.cuda, "Stream", lambda *a, **k: object())
    monkeypatch.setattr(torch.cuda, "stream", lambda s: contextlib.nullcontext())
    monkeypatch.setattr(torch.Tensor, "pin_memory", lambda self: self)
    from paper_1307_6488_b200 import replicas
    agg = replicas.aggregate_throughput                # its one-element timing tensor lives on "cuda" in bench.py
    monkeypatch.setattr(replicas, "aggregate_throughput", lambda s, u, dist=None, device="cpu": agg(s, u, dist, "cpu"))
    init = binding.Chemora.__init__

    def host_init(self, *a, **k):
        avail["v"] = False
        try:
            init(self, *a, **k)
        finally:
            avail["v"] = True

    monkeypatch.setattr(binding.Chemora, "__init__", host_init)
    binding.load()
    spec = importlib.util.spec_from_file_location("bench_emulated_mod", os.path.join(ROOT, "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def args(**kw):
    a = dict(gpus=1, steps=2, warmup=1, impl="ours", size=8, variant="auto", e2e_steps=2, cpu_sample=16, ref_sample=16,
             sweep=False, fill_floor=False, wave=False, wave1=False, paper_shape=False, ko_order=9,
             sweep_in_process=True, probe=False, probe_ids=0)
    a.update(kw)
    return types.SimpleNamespace(**a)


def last_json(capsys):
    out = capsys.readouterr().out.strip().splitlines()
    assert len([ln for ln in out if ln.startswith("{")]) == 1          # ONE JSON line
    return json.loads(out[-1])


@pytest.mark.parametrize("variant", ["auto", "0,1"])
def test_headline_run_prints_the_contract_line(bench, capsys, variant):
    bench.run_ours(args(variant=variant))
    line = last_json(capsys)
    base = json.load(open(os.path.join(ROOT, "BASELINE.json")))
    assert line["metric"] == base["metric"] and line["unit"] == "grid-point updates/s"
    for key in ("value", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline", "dtype",
                "data", "config", "roofline", "roofline_fp64", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert key in line, key
    assert line["steps"] == 2 and line["warmup"] == 1 and line["n_gpus"] == 1 and line["value"] > 0
    assert line["dtype"] == "f64" and line["data"] == "synthetic" and line["vs_baseline"] is None and line["scaling"] == "weak"
    cfg = line["config"]
    assert "workload" in cfg and "model" not in cfg and "l2" in cfg and cfg["multi_gpu"] == "replicas only"
    v = cfg["variant"]
    assert {"fused", "tile_id", "tile", "col_rows", "sweep_ms", "sweep_error"} <= set(v) and v["sweep_error"] is None
    assert (v["sweep_ms"] is not None) == (variant == "auto")
    r = line["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["traffic"] is None and r["peak"] > 0
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and r["step_frac"] > 0 and 0 < r["share_of_step"] <= 1.0001
    assert r["kernel"] == ("bssn_derivs+from_derivs" if variant == "0,1" else r["kernel"])
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] > 0 and "16^3" in cb["sample"]
    e = line["e2e"]
    nbytes = 25 * 8 ** 3 * 8
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == nbytes and e["d2h_bytes_per_step"] == nbytes
    # 2 timed steps: 4 fills + 4 right-hand sides each (split: two kernels per right-hand side)
    assert line["gpu_launches"] == 2 * (8 if variant == "auto" else 12)
    assert "sm_mhz" in line["clocks"] and "reasons" in line["clocks"]


def test_a_failing_sweep_does_not_cost_the_run(bench, capsys, monkeypatch):
    """chemora_autotune returning an error: bench falls back to the default fused tile and says so"""
    from paper_1307_6488_b200 import binding

    def boom(self):
        raise binding.ChemoraError(binding.ECUDA, "injected")

    monkeypatch.setattr(binding.Chemora, "autotune", boom)
    bench.run_ours(args())
    v = last_json(capsys)["config"]["variant"]
    assert v["fused"] == 1 and v["tile_id"] == 0 and "injected" in v["sweep_error"] and v["sweep_ms"] is None


def test_the_sweep_runs_in_a_child_by_default(bench, capsys, monkeypatch):
    """--variant auto without --sweep-in-process: `python bench.py --probe` in a child (a sticky device fault of a
    candidate then costs the sweep, not the headline run).  The child cannot be real here (it would load the real
    library and find no device), so subprocess.run is replaced by one that runs bench.run_probe in this process and
    hands back what it printed -- then by children that crash, print rubbish, or never end."""
    import subprocess
    seen = []

    def child(cmd, **kw):
        seen.append(cmd)
        assert cmd[1:] == [os.path.join(ROOT, "bench.py"), "--probe", "--size", "8"] and kw["timeout"] > 0
        bench.run_probe(args(probe=True))
        return types.SimpleNamespace(returncode=0, stdout="torch says hello\n" + capsys.readouterr().out, stderr="")

    monkeypatch.setattr(subprocess, "run", child)
    bench.run_ours(args(sweep_in_process=False))
    v = last_json(capsys)["config"]["variant"]
    assert len(seen) == 1 and v["sweep_process"] == "child" and v["sweep_error"] is None
    assert len(v["sweep_ms"]) == 18 and v["sweep_ms"][9 + v["tile_id"]] > 0 and v["fused"] == 1 and v["col_rows"] >= 1

    def crashed(cmd, **kw):
        return types.SimpleNamespace(returncode=-6, stdout="", stderr="a\nb\nCUDA error: an illegal memory access\nAborted")

    def rubbish(cmd, **kw):
        return types.SimpleNamespace(returncode=0, stdout='{"probe": {"fused": 1}}\n', stderr="")

    def endless(cmd, **kw):
        raise subprocess.TimeoutExpired(cmd, kw["timeout"])

    for fake, word in ((crashed, "illegal memory access"), (rubbish, "exit 0"), (endless, "no result within")):
        monkeypatch.setattr(subprocess, "run", fake)
        pick, err = bench.isolated_sweep(8)
        assert pick is None and word in err
    monkeypatch.setattr(subprocess, "run", crashed)                      # both children die: the default tile, said so
    bench.run_ours(args(sweep_in_process=False))
    line = last_json(capsys)
    v = line["config"]["variant"]
    assert (v["fused"], v["tile_id"], v["sweep_ms"], v["col_rows"]) == (1, 0, None, 32)
    assert v["sweep_error"].count("illegal memory access") == 2 and "bounded to fused ids 0..4" in v["sweep_error"]
    assert line["value"] > 0 and line["gpu_launches"] == 16

    # the unbounded child dies, the one bounded to the tiles of round 1 does not: its pick is used, and the line says so
    def second_time_lucky(cmd, **kw):
        if "--probe-ids" not in cmd:
            return crashed(cmd, **kw)
        assert cmd[-2:] == ["--probe-ids", "5"]
        bench.run_probe(args(probe=True, probe_ids=5))
        return types.SimpleNamespace(returncode=0, stdout=capsys.readouterr().out, stderr="")

    monkeypatch.setattr(subprocess, "run", second_time_lucky)
    bench.run_ours(args(sweep_in_process=False))
    v = last_json(capsys)["config"]["variant"]
    assert v["fused"] == 1 and v["tile_id"] < 5 and all(m == -1.0 for m in v["sweep_ms"][9 + 5:])
    assert "illegal memory access" in v["sweep_error"] and v["sweep_error"].endswith("fused ids 0..4: done")


def test_context_modes_run(bench, capsys, monkeypatch):
    from paper_1307_6488_b200 import inputs
    monkeypatch.setattr(inputs, "SWEEP_GRIDS", [(16, 4, 4)])
    bench.run_sweep(args())
    line = last_json(capsys)
    assert {(r["fused"], r["tile_id"]) for r in line["rows"]} == {(1, t) for t in range(8)} | {(0, t) for t in range(6)}
    assert all("sigma_model" in r for r in line["rows"] if r["fused"] and r["tile_id"] < 5) and len(line["tile_cost_model"]) == 1
    bench.run_fill_floor(args(size=8))
    line = last_json(capsys)
    assert [r["tile_id"] for r in line["rows"]] == list(range(8)) and all(r["fill_only_ms"] > 0 for r in line["rows"])
    bench.run_wave(args(size=16, wave=True))
    line = last_json(capsys)
    assert line["value"] > 0 and line["roofline"]["bound"] == "hbm"
