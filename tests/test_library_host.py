"""CPU-only tests of the product's host side: the C-ABI library loads and exports every symbol that
include/xc_b200.h declares; the host planner (host-only plan, device = -1) produces a valid plan; the
compute entry points fail loudly without a GPU; the N > 1 bench plumbing works over gloo (world_size 2)."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from workloads import make_workload

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def xc():
    from paper_2007_03143_b200 import build
    build.build()
    import paper_2007_03143_b200 as m
    return m


def test_library_exports_every_declared_symbol(xc):
    hdr = open(os.path.join(ROOT, "include", "xc_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(xc_[a-z_0-9]+)\s*\(", hdr))
    assert {"xc_plan_create", "xc_eval", "xc_integrate", "xc_plan_export", "xc_plan_destroy"} <= declared
    lib = C.CDLL(xc.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(xc.EXPORTED)


def test_no_cpu_fallback(xc):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    w = make_workload("c1")
    with pytest.raises(xc.XcError) as e:
        xc.Plan.from_workload(w)                     # device 0 without a GPU
    assert e.value.code == -4
    plan = xc.Plan.from_workload(w, device=-1)       # host-only plan: planner only
    from paper_2007_03143_b200 import binding as b
    E, N = C.c_double(), C.c_double()
    buf = np.zeros((25, 25))
    rc = b._lib.xc_eval(plan._h, buf.ctypes.data, 25, buf.ctypes.data, 25, C.byref(E), C.byref(N), 0, None)
    assert rc == -4
    rc = b._lib.xc_eval_host(plan._h, buf.ctypes.data, 25, buf.ctypes.data, 25, C.byref(E), C.byref(N), 0)
    assert rc == -4
    plan.close()


@pytest.mark.parametrize("name,max_pts", [("c1", 512), ("c1", 37), ("w8", 512), ("w27", 200), ("c2", 512)])
def test_host_planner_is_valid(xc, orc, name, max_pts):
    w = make_workload(name, with_P=False)
    plan = xc.Plan.from_workload(w, device=-1, max_batch_pts=max_pts)
    ex = plan.export()
    # the grid equals the oracle's canonical grid, point by point (same formulas, independent code)
    pts, wq, par = orc.build_grid(w.atoms_xyz, w.n_rad, w.n_ang)
    assert np.max(np.abs(pts[ex.orig] - ex.pts)) <= 1e-14 * np.max(np.abs(pts))
    assert np.max(np.abs(wq[ex.orig] - ex.wq)) <= 1e-14 * np.max(wq)
    assert np.array_equal(par[ex.orig], ex.parent)
    rc = orc.rcut(w.shell_nprim, w.shell_prim_off, w.exps)
    op = orc.Plan(ex.pts, ex.wq, ex.parent, ex.orig, ex.batch_off, ex.shell_off, ex.shells)
    assert orc.validate_plan(op, w.atoms_xyz, w.shell_atom, rc, max_pts) == 0      # Eq. (11), <= max_pts, S_j superset
    nq = np.diff(ex.batch_off)
    assert nq.min() >= 1 and nq.max() <= max_pts
    assert plan.algorithmic_flops == pytest.approx(orc.plan_flops(op, w.shell_L), rel=1e-12)
    if max_pts == 512 and name != "c1":
        assert np.mean(nq % 64 == 0) > 0.95      # almost every batch is a whole number of 64-point tiles
    plan.close()


def test_product_rule_and_bad_specs(xc):
    w = make_workload("c1", with_P=False)
    p = xc.Plan.from_workload(w, device=-1, spec=xc.grid_spec(10, 288, 0, angular=1))
    assert p.n_points == 3 * 10 * 288
    p.close()
    for bad in (xc.grid_spec(10, 287, 0, angular=1), xc.grid_spec(0, 26, 0), xc.grid_spec(10, 26, 3),
                xc.grid_spec(10, 26, 0, eta=0.0), xc.grid_spec(10, 26, 0, max_batch_pts=513)):
        with pytest.raises(xc.XcError) as e:
            xc.Plan.from_workload(w, device=-1, spec=bad)
        assert e.value.code == -1


def test_planner_is_deterministic(xc):
    w = make_workload("w8", with_P=False)
    a = xc.Plan.from_workload(w, device=-1).export()
    b = xc.Plan.from_workload(w, device=-1).export()
    assert np.array_equal(a.orig, b.orig) and np.array_equal(a.shells, b.shells) and np.array_equal(a.batch_off, b.batch_off)


def test_bench_reference_arm_and_gloo_two_ranks():
    # --impl reference prints one JSON line from rank 0; under world_size 2 the other rank exits 0 without work
    env = dict(os.environ, OMP_NUM_THREADS="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stderr
    import json
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0
    worker = os.path.join(ROOT, "tests", "gloo_worker.py")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29611", worker],
                         capture_output=True, text=True, timeout=600, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    assert "gloo ok 2" in out.stdout


def test_plan_does_not_depend_on_thread_count():
    """The planner bisects subtrees in parallel (OpenMP); the plan must be the same for any number of threads."""
    code = ("import hashlib, sys; sys.path.insert(0, %r)\n"
            "import paper_2007_03143_b200 as xc\n"
            "from workloads import make_workload\n"
            "w = make_workload('w27', with_P=False)\n"
            "p = xc.Plan.from_workload(w, spec=xc.grid_spec(w.n_rad, w.n_ang, 1), device=-1).export()\n"
            "print(hashlib.sha1(p.orig.tobytes() + p.batch_off.tobytes() + p.shell_off.tobytes() + p.shells.tobytes()).hexdigest())\n"
            % ROOT)
    digests = []
    for n in ("1", "3", "8"):
        env = dict(os.environ, OMP_NUM_THREADS=n)
        out = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, check=True).stdout.strip()
        digests.append(out)
    assert len(set(digests)) == 1 and len(digests[0]) == 40
