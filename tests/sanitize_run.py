"""Small runs of every kernel path for compute-sanitizer ("race detection / sanitizers"):

    compute-sanitizer --tool memcheck  python tests/sanitize_run.py
    compute-sanitizer --tool racecheck python tests/sanitize_run.py

Not a pytest file: it only drives the library (no oracle) and checks the weight balance of each run, so that the
sanitizer sees the history kernel (analog, weighted, census-step and generation variants, staged and unstaged tables,
pools forced to overflow into the global fission ring queue, general CSG regions, a lattice), the census-stepped
kernels, the control kernels and the close-out on problems that finish in seconds under instrumentation."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import paper_2409_04668_b200 as M  # noqa: E402
from workloads import configs as W  # noqa: E402

N = int(os.environ.get("MCDC_SANITIZE_N", "6000"))


def balance(c):
    lhs = c["source"] + c["production"] + c["vr_gain"]
    rhs = c["capture"] + c["fission_abs"] + c["leak"] + c["census_final"] + c["lost"] + c["vr_loss"]
    assert abs(lhs - rhs) <= 1e-9 * max(1.0, lhs), (lhs, rhs)


def run(name, p, tech=None, eigen=False, **opts):
    g = M.Problem(p)
    if tech:
        g.set_technique(**tech)
    if eigen:
        g.run_eigenvalue(p.n_histories, p.seed, 1, 2)
    else:
        g.run(**opts)
    c = g.counters()
    if not eigen:                                          # (generations are renormalised between them: no run-wide balance)
        balance(c)
    print(f"{name:34s} {g.kernel_info().split(' grid')[0]:40s} segments {c['segments']:9d} launches {c['kernel_launches']}")
    g.tallies()
    g.close()


def main():
    pc = dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0, population_control=True)
    ic = dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0)
    run("config0 analog", W.config0_infinite_medium(n_histories=N, n_batches=4))
    run("config1 analog, general scorer", W.config1_slab(n_histories=N, n_batches=4))
    run("config3 analog", W.config3_pin_lattice(n_histories=N, n_batches=4))
    run("config3 record, queue forced", W.config3_pin_lattice(n_histories=N, n_batches=4), record_history_events=True,
        debug_pool_slots=32)
    run("config3 unstaged tables", W.config3_pin_lattice(n_histories=N, n_batches=4), debug_stage_tables=-1)
    run("config3 weighted", W.config3_pin_lattice(n_histories=N, n_batches=4), tech=ic)
    run("config3 census-step + control", W.config3_pin_lattice(n_histories=N, n_batches=4), tech=pc)
    run("config3 k-eigenvalue", W.as_eigenvalue(W.config3_pin_lattice(n_histories=N, n_batches=1)), eigen=True)
    run("stress geometry", W.stress_geometry(n_histories=N, n_batches=4))
    run("csg regions", W.csg_union_geometry(n_histories=N, n_batches=4))
    run("csg regions + control", W.csg_union_geometry(n_histories=N, n_batches=4), tech=pc)
    run("mixed lattice", W.lattice_mixed(n_histories=N, n_batches=4))
    run("config1 census-stepped kernel", W.config1_slab(n_histories=N, n_batches=4), scheduler=1)
    run("config3 census-stepped + control", W.config3_pin_lattice(n_histories=N, n_batches=4), tech=pc, scheduler=1)
    print("sanitize_run: all balances closed")


if __name__ == "__main__":
    main()
