"""CPU-only checks of the host logic around the CUDA path: the C-ABI library loads and exports every symbol
include/mfc_b200.h declares (no compute call — there is no GPU here), bench.py's metric arithmetic, the
algorithmic flop counts its roofline line uses (re-derived with the operation-counting oracle), and the N > 1
launch path (world_size 2, gloo)."""
import ctypes
import dataclasses
import json
import os
import re
import subprocess
import sys

import numpy as np
import pytest

import mfc_workloads as W
from oracle import oracle as O

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    with open(os.path.join(ROOT, "include", "mfc_b200.h")) as f:
        text = re.sub(r"/\*.*?\*/", "", f.read(), flags=re.S)
    return sorted(set(re.findall(r"\b(mfc_[a-z0-9_]+)\s*\(", text)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    import paper_2503_07953_b200 as M
    from paper_2503_07953_b200 import build as B
    path = B.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    names = declared_symbols()
    assert {"mfc_init_grid", "mfc_prim_from_cons", "mfc_rhs", "mfc_rk3_step", "mfc_cfl_dt"} <= set(names)
    for name in names:
        assert hasattr(lib, name), name
    assert set(M.EXPORTS) == set(names), set(M.EXPORTS) ^ set(names)


def test_product_package_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2503_07953_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                with open(os.path.join(dirpath, fn)) as f:
                    text = f.read()
                assert "oracle" not in text.replace("shares nothing with oracle/", "").replace(
                    "the CPU oracle is written separately", ""), fn
    with open(os.path.join(ROOT, "mfc_workloads", "__init__.py")) as f:
        text = f.read()
    assert "import oracle" not in text and "from oracle" not in text and "paper_2503_07953_b200" not in text


def test_no_cpu_fallback_without_cuda():
    import torch
    import paper_2503_07953_b200 as M
    if torch.cuda.is_available():
        pytest.skip("needs a machine without a GPU")
    case = W.config(1, n=32)
    with pytest.raises(RuntimeError):
        M.Grid.from_case(case)
    # straight through the C ABI: no usable device -> an error status, never a result
    p = M.MfcParams()
    p.ndim, p.nfluids = 1, 1
    gam, pi = (ctypes.c_double * 1)(1.4), (ctypes.c_double * 1)(0.0)
    p.gamma = ctypes.cast(gam, ctypes.POINTER(ctypes.c_double))
    p.pi_inf = ctypes.cast(pi, ctypes.POINTER(ctypes.c_double))
    for d in range(3):
        p.n[d], p.dx[d], p.bc_lo[d], p.bc_hi[d] = (32 if d == 0 else 1), 1.0, 1, 1
    p.weno_eps, p.alpha_floor, p.clamp, p.device = 1e-16, 1e-6, 1, 0
    h = ctypes.c_void_p()
    st = M.lib().mfc_init_grid(ctypes.byref(p), ctypes.byref(h))
    assert st in (M.MFC_ERR_CUDA, M.MFC_ERR_ARG) and not h.value
    assert M.lib().mfc_last_error()


def test_grind_time_arithmetic():
    import bench
    # 3 RHS evaluations per step: 10 steps of 1e6 cells x 8 equations in 24 ms -> 0.1 ns
    assert bench.grind_ns(24.0, 10, 10 ** 6, 8) == pytest.approx(0.1)
    assert bench.grind_ns(24.0, 10, 10 ** 6, 8, replicas=2) == pytest.approx(0.05)
    assert bench.sweep_alg_bytes_per_cell("sweep_x", 8, 3) == 128
    assert bench.sweep_alg_bytes_per_cell("sweep_y", 8, 3) == 192           # middle sweep: q and L read, L written
    assert bench.sweep_alg_bytes_per_cell("sweep_z", 8, 3) == pytest.approx(8 * (24 + 32 + 32) / 3)  # last sweep + RK stage, mean of 3
    assert bench.sweep_alg_bytes_per_cell("sweep_y", 7, 2) == pytest.approx(7 * (24 + 32 + 32) / 3)
    # algorithmic bytes of an RK stage, whatever the design: 576 B per cell per step at neq = 8 with the CFL read
    assert 3 * bench.stage_alg_bytes_per_cell(8) + 8 * 8 == 576
    assert len(bench.kernel_sources_sha256()) == 64
    assert bench.median([3.0, 1.0, 2.0]) == 2.0 and bench.median([4.0, 1.0, 2.0, 3.0]) == 2.5
    assert bench.FP64_PEAK_TFLOPS_DERIVED == pytest.approx(37.225, rel=1e-3)


@pytest.mark.parametrize("weno", ["js", "m", "z"])
@pytest.mark.parametrize("index,n", [(1, 400), (2, 400), (3, 48), (4, 16), (5, 16)])
def test_algorithmic_flops_per_cell_match_the_operation_counting_oracle(index, n, weno):
    """bench.ALG_FLOPS_PER_CELL_RHS is the n -> infinity value of (add + mul + div + sqrt)/cells.  One face more
    than cells per line is solved, so the count on n cells per direction is  A + B/n  exactly; two sizes fix A."""
    import bench

    def per_cell(m):
        case = dataclasses.replace(W.config(index, n=m), weno=weno)
        c = O.Oracle(case).count_rhs(W.initial_state(case))
        return (c["add"] + c["mul"] + c["div"] + c["sqrt"]) / case.cells

    f1, f2 = per_cell(n), per_cell(2 * n)
    a = 2 * f2 - f1  # f(n) = A + B/n
    assert a == pytest.approx(bench.ALG_FLOPS_PER_CELL_RHS_BY_WENO[weno][index], rel=2e-3), (f1, f2, a)


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "rhs_grind_time" and line["higher_is_better"] is False
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"] > 0


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.reduce_max_ms(10.0 + 5.0 * rank, world)          # slowest rank decides
val = bench.grind_ns(ms, 4, 1000, 8, world)                 # whole-job aggregate over the replicas
print(json.dumps({{"rank": rank, "ms": ms, "val": val}}))
dist.destroy_process_group()
"""


def test_replica_launch_path_world_size_2_gloo(tmp_path):
    """N > 1 is 'replicas only': no data-path collective; the only exchange is the max over ranks
    of the device time.  Two gloo ranks must agree on it and on the aggregate value."""
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29577", str(script)],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    # the two ranks write to one pipe: their lines may arrive glued together
    recs = [json.loads(m) for m in re.findall(r"\{[^{}]*\}", out.stdout)]
    assert sorted(r["rank"] for r in recs) == [0, 1]
    for r in recs:
        assert r["ms"] == 15.0
        assert r["val"] == pytest.approx(15.0 * 1e6 / (3 * 4 * 1000 * 8 * 2))


# ------------------------------------------------------------------ slab decomposition: host logic and the exchange over gloo
def test_slab_partition_neighbours_and_local_case():
    from paper_2503_07953_b200 import slab as S
    import paper_2503_07953_b200 as M
    assert S.partition(10, 3) == [(0, 4), (4, 3), (7, 3)]
    assert sum(c for _, c in S.partition(257, 8)) == 257
    with pytest.raises(ValueError):
        S.partition(8, 3)                                   # a slab of 2 cells cannot fill a 3-deep halo
    assert S.neighbours(0, 4, True) == (3, 1) and S.neighbours(3, 4, True) == (2, 0)
    assert S.neighbours(0, 4, False) == (None, 1) and S.neighbours(3, 4, False) == (2, None)
    assert S.neighbours(0, 1, True) == (0, 0) and S.neighbours(0, 1, False) == (None, None)
    case = W.config(5, n=24)                                # extrapolation on every side
    c0, s0, n0 = S.local_case(case, 0, 3)
    c2, s2, n2 = S.local_case(case, 2, 3)
    assert (s0, n0, s2, n2) == (0, 8, 16, 8) and c0.n == (24, 24, 8) and c0.dx == case.dx
    assert c0.bc_lo[2] == M.BC_EXTRAP and c0.bc_hi[2] == M.BC_HALO and c2.bc_lo[2] == M.BC_HALO and c2.bc_hi[2] == M.BC_EXTRAP
    assert c0.bc_lo[:2] == case.bc_lo[:2]
    cp, _, _ = S.local_case(W.config(4, n=24), 1, 2)        # periodic: halos on both ends of every slab
    assert cp.bc_lo[2] == M.BC_HALO and cp.bc_hi[2] == M.BC_HALO
    with pytest.raises(ValueError):
        S.local_case(W.config(1), 0, 2)                     # 1-D


_SLAB_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2503_07953_b200 import slab as S
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
res = dict(rank=rank)
for periodic in (True, False):
    below, above = S.neighbours(rank, world, periodic)
    mk = lambda v: torch.full((12,), float(v), dtype=torch.float64)
    send_lo, send_hi = mk(10 * rank + 1), mk(10 * rank + 2)
    halo_lo = mk(-1) if below is not None else None
    halo_hi = mk(-1) if above is not None else None
    S.exchange(send_lo if below is not None else None, send_hi if above is not None else None, halo_lo, halo_hi,
               rank, below, above, dist, None)
    res["p" if periodic else "e"] = [None if halo_lo is None else halo_lo.tolist(), None if halo_hi is None else halo_hi.tolist(),
                                     below, above]
    t = torch.tensor([1.0 + rank]); dist.all_reduce(t, op=dist.ReduceOp.MIN); res["min"] = float(t)
print(json.dumps(res))
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world", [2, 3])
def test_slab_exchange_over_gloo(tmp_path, world):
    """every slab receives its lower neighbour's top layers as halo_lo and its upper neighbour's bottom layers as halo_hi —
    also when both neighbours are the same peer (two slabs, periodic), where only the posting order tells the two
    messages apart"""
    script = tmp_path / "slab_worker.py"
    script.write_text(_SLAB_WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
                          "--master-addr", "127.0.0.1", "--master-port", str(29580 + world), str(script)],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    recs = {}
    for l in out.stdout.replace("}{", "}\n{").splitlines():
        if l.startswith("{"):
            r = json.loads(l)
            recs[r["rank"]] = r
    assert sorted(recs) == list(range(world))
    for rank, r in recs.items():
        assert r["min"] == 1.0
        for key in ("p", "e"):
            lo, hi, below, above = r[key]
            if below is None:
                assert lo is None
            else:
                assert lo == [10.0 * below + 2] * 12          # the lower neighbour's send_hi
            if above is None:
                assert hi is None
            else:
                assert hi == [10.0 * above + 1] * 12          # the upper neighbour's send_lo
        assert r["p"][2] == (rank - 1) % world and r["p"][3] == (rank + 1) % world
