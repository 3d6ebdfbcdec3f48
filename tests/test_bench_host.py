"""Host logic of bench.py that needs no GPU: `--gpus N` starts N ranks by itself (the multi-GPU command),
the reference arm prints ONE line from rank 0, the ncu constants are only handed out for the kernel build they were
captured from, and the all-cores CPU baseline covers disjoint history ranges."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_bench_gpus_2_launches_two_ranks_itself_and_rank0_prints_one_line():
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--ref-seconds", "0.2", "--workload", "config0"],
                       capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2            # the real world size, not the flag
    assert d["config"]["histories_per_step"] < d["config"]["workload_histories"]   # the sample size is stated
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_ncu_constants_are_keyed_by_kernel_workload_and_revision():
    import bench
    with open(bench.NCU_JSON) as f:
        cap = json.load(f)["captures"][0]
    info = f"{cap['kernel']} rev={cap['rev']} grid=148 pool_slots=104 smem=1"
    e, note = bench.ncu_constants(info, cap["workload"], cap.get("technique", "analog"))
    assert e is not None and e["thread_inst_per_segment"] > 0 and note == cap["source"]
    assert os.path.exists(os.path.join(ROOT, cap["source"]))
    e, note = bench.ncu_constants(info.replace(cap["rev"], "0" * 12), cap["workload"], "analog")
    assert e is None and "stale" in note
    e, note = bench.ncu_constants(info, "config2_shield_duct", "analog")
    assert e is None
    e, note = bench.ncu_constants("", cap["workload"], "analog")
    assert e is None
    # a later entry of the same kernel / workload whose revision matches is found, not reported stale at the first name match
    with open(bench.NCU_JSON) as f:
        caps = json.load(f)["captures"]
    older = [c for c in caps[1:] if (c["kernel"], c["workload"], c.get("technique", "analog")) ==
             (cap["kernel"], cap["workload"], cap.get("technique", "analog")) and c["rev"] != cap["rev"]]
    if older:
        e, note = bench.ncu_constants(info.replace(cap["rev"], older[0]["rev"]), cap["workload"], cap.get("technique", "analog"))
        assert e is not None and e["rev"] == older[0]["rev"] and note == older[0]["source"]


def test_kernel_revision_covers_the_host_file_and_the_defines_and_tuned_builds_go_elsewhere():
    from paper_2409_04668_b200 import build as b
    assert b.kernel_rev() == b.kernel_rev([]) and len(b.kernel_rev()) == 12
    assert b.kernel_rev(["-DMCDC_WARP_THREADS=576"]) != b.kernel_rev()
    assert b.kernel_rev(["-DA=1", "-DB=2"]) == b.kernel_rev(["-DB=2", "-DA=1"]) != b.kernel_rev(["-DA=1"])
    assert b.LIB_TUNED != b.LIB and b.OBJ_TUNED != b.OBJ and b.lib_path() == b.LIB
    src = open(os.path.join(ROOT, "paper_2409_04668_b200", "build.py")).read()
    assert '"mcdc_host.cu"]' in src.split("def kernel_rev")[1].split("def ")[0]


def test_algorithmic_bytes_formula():
    """176 B per segment + 112 B per fission child + 88 B per source history (history kernel only)."""
    import bench
    assert bench.algorithmic_bytes(None, {"segments": 10, "children": 2}, 3) == 1760 + 224 + 264


def test_all_cores_cpu_baseline_runs_one_process_per_core():
    import argparse

    import bench
    from workloads import configs as W
    args = argparse.Namespace(workload="config0", histories=0, batches=0)
    p = W.get_config("config0")
    out = bench.run_cpu_all_cores(args, p, per_core_rate=2000.0, seconds_target=0.5)
    assert out["cores"] == (os.cpu_count() or 1) and out["kind"] == "oracle"
    assert out["value"] > 0 and f"{out['cores']} processes" in out["sample"]
