"""Host-side logic of bench.py's N > 1 path ("replicas only") under gloo with world_size 2:
max-over-ranks timing, whole-job value, and the reference arm printing on rank 0 only."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")
    out[rank] = (ms, bench.job_value(100, 3, world, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_job_value_world_size_2():
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, 29731, out), nprocs=2, join=True)
        res = dict(out)
    assert res[0] == res[1]
    ms, value = res[0]
    assert ms == 15.0                                    # the slower rank decides
    assert abs(value - 2 * 100 * 3 / 15e-3) < 1e-6       # aggregate over both replicas


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "cfg1",
                        "--gpus", "2", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "cfg1",
                        "--gpus", "2", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0


# ---- NEXT-2 host logic: the spinor index sharded over ranks, densities summed with a real collective (gloo) ----------
def _shard_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import numpy as np
    import workloads as wl
    from harness import make_oracle
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = wl.cfg3(n_side=8, n_kz=3, nz=8, n_steps=1)          # 192 spinors in 3 k_z modes (multiplicity 1, 2, 2)
    n0, n1 = wl.shard_range(w.n_wf, rank, world)
    ws_ = wl.shard(w, n0, n1)
    psi = ws_.spinors()                                      # this rank's spinors only
    o = make_oracle(ws_)
    o.densities(psi)
    red = {}
    for f in ("rho_a", "rho_b", "nu"):                       # densities as the functional sees them (linear in the sums)
        loc = np.ascontiguousarray(o.get_field(f))
        t = torch.from_numpy(loc.view(np.float64).copy())
        dist.all_reduce(t)                                   # the one exchange of the sharded step
        red[f] = t.numpy().view(loc.dtype).reshape(loc.shape)
    assert w.spin_symmetric                                  # get_field folds (rho_a + rho_b, 2 nu): undo it for the raw sums
    o.set_field("rho_a", red["rho_a"]); o.set_field("rho_b", np.zeros_like(red["rho_b"])); o.set_field("nu", 0.5 * red["nu"])
    o.update_potentials()
    out[rank] = (n0, n1, red, {f: np.array(o.get_field(f)) for f in ("delta", "U_a", "U_b")},
                 np.array_equal(psi, w.spinors(n0, n1)))
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_densities_and_potentials_world_size_2():
    """Each rank builds the densities of its own share of the spinors (mode table shifted and clipped, a k_z mode cut
    in two), one all-reduce sums them, and every rank then forms the same potentials as the unsharded problem."""
    import numpy as np
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import workloads as wl
    from harness import make_oracle, relerr
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_shard_worker, args=(2, 29733, out), nprocs=2, join=True)
        res = dict(out)
    w = wl.cfg3(n_side=8, n_kz=3, nz=8, n_steps=1)
    assert (res[0][0], res[0][1], res[1][0], res[1][1]) == (0, w.n_wf // 2, w.n_wf // 2, w.n_wf)
    assert res[0][4] and res[1][4]                           # a shard generates exactly its slice of the spinors
    o = make_oracle(w)
    o.densities(w.spinors())
    o.update_potentials()
    for r in (0, 1):
        for f in ("rho_a", "rho_b", "nu"):
            assert relerr(res[r][2][f], o.get_field(f)) < 1e-13, f
        for f in ("delta", "U_a", "U_b"):
            assert relerr(res[r][3][f], o.get_field(f)) < 1e-12, f
    assert all(np.array_equal(res[0][3][f], res[1][3][f]) for f in ("delta", "U_a", "U_b"))   # ranks agree bit for bit


def test_shard_ranges_cover_the_spinor_index():
    sys.path.insert(0, ROOT)
    import workloads as wl
    for n_wf, world in ((16384, 8), (10, 3), (7, 8), (262144, 4)):
        r = [wl.shard_range(n_wf, k, world) for k in range(world)]
        assert r[0][0] == 0 and r[-1][1] == n_wf and all(r[k][1] == r[k + 1][0] for k in range(world - 1))
        assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1
