"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/ocgs.h declares (no compute calls),
host-only helpers behave, and the N > 1 view sharding + statistics merge works over gloo with world_size 2."""
import ctypes
import os
import re
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2501_08174_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "ocgs.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ocgs(?:3d)?_[a-z0-9_]+)\s*\(", hdr))
    assert {"ocgs_preprocess", "ocgs_bin_sort", "ocgs_render_fwd", "ocgs_render_bwd", "ocgs_prune_stats"} <= declared
    for name in sorted(declared):
        assert hasattr(lib, name), name
    from paper_2501_08174_b200 import binding
    assert set(binding.EXPORTS) <= declared


def test_default_config_and_workspace_layout(lib):
    from paper_2501_08174_b200 import binding as B
    cfg = B.ocgs_config()
    lib.ocgs_default_config(ctypes.byref(cfg))
    assert cfg.tile == 16 and cfg.sh_degree == 3 and abs(cfg.near_z - 0.2) < 1e-7 and cfg.rho_max == 9.0
    assert cfg.alpha_min == np.float32(1.0 / 255.0) and abs(cfg.alpha_max - 0.99) < 1e-7 and cfg.filter_sigma2 == 0.5
    assert abs(cfg.gamma_bg - 0.5) < 1e-7 and cfg.tau_contrib == 0.0 and cfg.min_opacity == 0.0  # gamma: PAPER.md:129
    L = B.ocgs_ws_layout()
    assert lib.ocgs_workspace_layout(1000, 1920, 1080, ctypes.c_size_t(50_000), ctypes.byref(L)) == 0
    offs = [getattr(L, f) for f in B._LAYOUT_FIELDS[1:]]
    assert offs == sorted(offs) and all(o % 256 == 0 for o in offs) and L.total_bytes > offs[-1]
    assert L.rec - L.rank_to_id >= 4 * 1000 and L.tile_vals - L.tile_keys >= 4 * 50_000
    lib.ocgs_workspace_bytes.restype = ctypes.c_size_t
    assert lib.ocgs_workspace_bytes(1000, 1920, 1080, ctypes.c_size_t(50_000)) == L.total_bytes
    # over the limits -> OCGS_ERR_UNSUPPORTED / 0 bytes
    assert lib.ocgs_workspace_layout(10, 40000, 100, ctypes.c_size_t(10), ctypes.byref(L)) == -4
    assert lib.ocgs_workspace_bytes(10, 100, 100, ctypes.c_size_t(1 << 33)) == 0
    # null arguments are rejected before any CUDA call
    assert lib.ocgs_preprocess(None, None, None, None, ctypes.c_size_t(0), None) == -1


def test_views_for_rank_partitions_views():
    from paper_2501_08174_b200.sharding import views_for_rank
    for n_views, world in ((49, 8), (64, 4), (3, 8), (16, 1)):
        got = sorted(v for r in range(world) for v in views_for_rank(n_views, r, world))
        assert got == list(range(n_views))
    with pytest.raises(ValueError):
        views_for_rank(4, 2, 2)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import oracle as orc
    from paper_2501_08174_b200 import scenegen as sg
    from paper_2501_08174_b200.sharding import allreduce_stats, views_for_rank
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sc = sg.make_scene("config1", n_obj=300, n_bg=100, res=48, f=56.0)
    cfg = orc.default_config(sh_degree=0)
    vis = np.zeros(sc.n, np.uint32)
    cs = np.zeros(sc.n, np.float64)
    for v in views_for_rank(len(sc.cameras), rank, world):
        cam = orc.camera_from(sc.cameras[v])
        pre = orc.preprocess(sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh, cam, cfg)
        srt = orc.bin_sort(pre, cam, cfg)
        orc.render_fwd(pre, srt, sc.opacity, cam, cfg, vis_count=vis, contrib_sum=cs, want_fragile=False)
    tv, tc = torch.tensor(vis.astype(np.int64)), torch.tensor(cs)
    allreduce_stats(tv, tc)
    q.put((rank, tv.numpy(), tc.numpy()))
    dist.barrier()
    dist.destroy_process_group()


def test_statistics_merge_over_gloo_world2_matches_single_process():
    import torch.multiprocessing as mp
    import oracle as orc
    from paper_2501_08174_b200 import scenegen as sg
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 500)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=180) for _ in procs]
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    sc = sg.make_scene("config1", n_obj=300, n_bg=100, res=48, f=56.0)
    cfg = orc.default_config(sh_degree=0)
    vis = np.zeros(sc.n, np.uint32)
    cs = np.zeros(sc.n, np.float64)
    for v in range(len(sc.cameras)):
        cam = orc.camera_from(sc.cameras[v])
        pre = orc.preprocess(sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh, cam, cfg)
        srt = orc.bin_sort(pre, cam, cfg)
        orc.render_fwd(pre, srt, sc.opacity, cam, cfg, vis_count=vis, contrib_sum=cs, want_fragile=False)
    for rank, tv, tc in res:
        assert np.array_equal(tv, vis.astype(np.int64))
        assert np.allclose(tc, cs, rtol=1e-12, atol=1e-15)
    # every rank derives the same prune mask from the merged statistics (replicas stay in lock-step)
    m0 = orc.prune(res[0][1].astype(np.uint32), res[0][2].astype(np.float32), sc.opacity)["prune_mask"]
    m1 = orc.prune(res[1][1].astype(np.uint32), res[1][2].astype(np.float32), sc.opacity)["prune_mask"]
    assert np.array_equal(m0, m1)


def _bench_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from paper_2501_08174_b200 import sharding
    assert sharding.env_rank() == (rank, world, rank)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    views = sharding.rotation_for_rank(49, rank, world, 8)
    # every rank "measures" its own step time; the bench reports the max over ranks and the whole-job aggregate
    ms_local = 2.0 + rank
    ms = sharding.max_over_ranks(ms_local)
    grads = dict(d_pos=torch.full((5, 3), float(rank + 1)), d_sh=torch.full((5, 16, 3), 10.0 * (rank + 1)))
    nbytes = sharding.allreduce_grads(grads)
    q.put((rank, views, ms, nbytes, float(grads["d_pos"][0, 0]), float(grads["d_sh"][0, 0, 0]),
           sharding.aggregate_throughput(1_000_000, world, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_bench_rank_bookkeeping_over_gloo_world2():
    """bench.py's own multi-rank bookkeeping (paper_2501_08174_b200.sharding), on two gloo ranks: view rotation per rank, max over
    ranks of the measured time, whole-job aggregate, and the gradient all-reduce of the batched-view mode."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + (os.getpid() % 500)
    procs = [ctx.Process(target=_bench_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert res[0][1] == [0, 2, 4, 6, 8, 10, 12, 14] and res[1][1] == [1, 3, 5, 7, 9, 11, 13, 15]
    for rank, views, ms, nbytes, gp, gs, thr in res:
        assert ms == 3.0                        # max over ranks
        assert nbytes == (15 + 240) * 4
        assert gp == 3.0 and gs == 30.0         # sum over ranks
        assert thr == pytest.approx(2 * 1_000_000 / 3.0e-3)


def test_view_rotation_and_launcher_rules():
    from paper_2501_08174_b200 import sharding
    assert sharding.rotation_for_rank(49, 0, 1, 8) == list(range(8))
    assert sharding.rotation_for_rank(49, 3, 8, 0) == [3, 11, 19, 27, 35, 43]
    assert sorted(v for r in range(8) for v in sharding.rotation_for_rank(49, r, 8, 0)) == list(range(49))  # a partition
    assert sharding.rotation_for_rank(4, 6, 8, 2) == [2]                                                  # more ranks than views
    assert sharding.relaunch_under_torchrun(1, ["x"], available=0) is None
    with pytest.raises(RuntimeError, match="needs 2 CUDA devices"):
        sharding.relaunch_under_torchrun(2, ["x"], available=1)


def test_bench_refuses_more_gpus_than_the_node_has():
    """`python bench.py --gpus N` starts the N ranks itself; on a node with fewer CUDA devices it must fail loudly rather than
    measure fewer GPUs than it names (here: any N above the number of devices present)."""
    import subprocess
    import torch
    n = (torch.cuda.device_count() if torch.cuda.is_available() else 0) + 1
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", str(max(n, 2))], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode != 0 and f"needs {max(n, 2)} CUDA devices" in r.stderr


def test_defaults_match_the_constants_the_paper_states():
    """tests/golden/paper_constants.txt: gamma = 0.5 in the library's default config (through the C ABI: the
    helper is host-only) and in the oracle's; the pruning intervals are the training loop's business and only recorded."""
    import os
    import oracle as orc
    from paper_2501_08174_b200 import binding as B
    vals = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")):
        if line.strip() and not line.startswith("#"):
            name, value = line.split()[:2]
            vals[name] = float(value)
            assert "PAPER.md:" in line
    assert B.ocgs_default_config().gamma_bg == vals["gamma_bg"] == orc.default_config().gamma_bg
    assert (vals["prune_interval_dtu"], vals["prune_interval_mipnerf360"], vals["iterations"]) == (100, 600, 30000)
