"""CPU-side tests of the boundary and the host logic (no compute calls without a GPU): the shared library builds,
loads and exports every symbol include/sps.h declares; ctypes mirrors of the ABI structs have the C layout; the
library refuses to compute without an sm_100 device (no CPU fallback); seeded workloads are reproducible; the
multi-rank plumbing works over gloo with world_size 2."""
import ctypes as C
import os
import re
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as G
    G.build()
    from paper_2506_19919_b200 import binding
    return binding.lib()


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "sps.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(sps_[a-z0-9_]+)\s*\(", hdr))
    assert {"sps_create_table", "sps_photometry", "sps_loglike_grad", "sps_hmc_run"} <= names
    for n in sorted(names):
        assert hasattr(lib, n), n
    from paper_2506_19919_b200 import binding
    assert set(binding.EXPORTS) <= names


def test_struct_layouts_match_the_header():
    from paper_2506_19919_b200 import binding as b
    # 5 int32 (+pad), 6 pointers, 5 doubles, 2 int32, 3 pointers, double, int32 (+pad), 2 pointers
    assert C.sizeof(b._TableDesc) == 5 * 4 + 4 + 6 * 8 + 5 * 8 + 2 * 4 + 3 * 8 + 8 + 4 + 4 + 2 * 8
    assert b._TableDesc.model.offset == 116 and b._TableDesc.filt_wave_A.offset == 120 and b._TableDesc.gauss_mu.offset == 160
    assert C.sizeof(b._Prior) == 7 * 8
    assert C.sizeof(b._HmcConfig) == 7 * 4 + 2 * 4 + 4 + 8 + 4 + 4 + 3 * 8  # 7 int32, 2 float, pad, uint64, uint32, pad, 3 pointers
    assert b._HmcConfig.seed.offset == 40
    assert C.sizeof(b._HmcSummary) == 11 * 8


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2506_19919_b200 import binding, workloads as W
    with pytest.raises(binding.SpsError) as e:
        binding.sps_create_table(W.make_grid("tiny"))
    assert "status 5" in str(e.value)                                   # SPS_EUNSUPPORTED
    assert lib.sps_launch_count() == 0


def test_bad_descriptor_is_rejected_before_touching_the_device(lib):
    from paper_2506_19919_b200 import binding as b
    h = C.c_void_p()
    assert lib.sps_create_table(None, C.byref(h)) == 1                  # SPS_EINVAL
    assert b"null" in lib.sps_last_error()
    d = b._TableDesc()                                                  # all-null arrays
    assert lib.sps_create_table(C.byref(d), C.byref(h)) == 1


def test_workloads_are_seeded_and_shaped():
    from paper_2506_19919_b200 import workloads as W
    g1, g2 = W.make_grid("tiny"), W.make_grid("tiny")
    assert g1.ssp.shape == (80, 500) and g1.ssp.dtype == np.float32 and (g1.ssp > 0).all()
    assert np.array_equal(g1.ssp, g2.ssp)
    p = W.make_prior()
    a, b = W.draw_theta_unbounded(p, 16, 7), W.draw_theta_unbounded(p, 16, 7)
    assert a.shape == (16, 13) and np.array_equal(a, b)
    assert not np.array_equal(a, W.draw_theta_unbounded(p, 16, 8))
    assert set(W.CONFIGS) == {"c1_tiny_hmc", "c2_exact", "c3_approx", "c4_hmc", "c5_nuts"}


def test_galaxy_shards_partition_the_catalogue():
    from paper_2506_19919_b200.sharding import galaxy_shard
    for n, w in ((10000, 8), (7, 3), (5, 8), (0, 2)):
        spans = [galaxy_shard(n, r, w) for r in range(w)]
        assert spans[0][0] == 0 and spans[-1][1] == n
        assert all(spans[i][1] == spans[i + 1][0] for i in range(w - 1))
        sizes = [b - a for a, b in spans]
        assert max(sizes) - min(sizes) <= 1


def _gloo_worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sys.path.insert(0, ROOT)
    from paper_2506_19919_b200.sharding import aggregate_throughput, galaxy_shard, max_over_ranks, rank_seed
    a, b = galaxy_shard(101, rank, world)
    t_dev, t_e2e = max_over_ranks([1.0 + rank, 3.0 - rank], dist)       # every rank must see the slowest rank's time
    out[rank] = (a, b, rank_seed(5, rank), t_dev, t_e2e, aggregate_throughput(50.0, world, t_dev))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_timing_reduction_over_gloo():
    import torch.multiprocessing as mp
    world, port = 2, 29500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_gloo_worker, args=(world, port, out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    assert (r0[0], r0[1], r1[0], r1[1]) == (0, 51, 51, 101)
    assert r0[2] != r1[2]
    assert r0[3] == r1[3] == 2.0 and r0[4] == r1[4] == 3.0
    assert r0[5] == r1[5] == 50.0
