"""N > 1 host logic on CPU: world_size 2, gloo.  Each rank searches its band of start rows of one
replicated stack through shard.search_row_band, whose per-rank search is the PRODUCT's band call
(launch_search_tiled with y_begin / y_end, the code behind kbmod_search_rows) run under the SIMT
emulator of tests/hostlogic/ in place of a GPU; the concatenated planes must equal the oracle's
single-process search bit for bit, and the step time must be the slowest rank's."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1901_02492_b200 import shard, synth


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, ret):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert shard.world() == (rank, world)
        pp = synth.random_psiphi(4, 23, 40, seed=11, invalid_frac=0.05)     # same stack on every rank
        vel = synth.velocity_grid(4, 3, -1.0, 1.0, 2.0, 9.0)
        times = [0.0, 0.4, 1.0, 1.5]
        from tests import simt_build, test_tiled_simt as T
        sim = simt_build.load("tiled_simt")

        def emulated_search(psiphi, times, vel_grid, K, min_obs, y_begin, y_end):
            out = T.run_sim(sim, psiphi.numpy(), times, vel_grid, K, min_obs, T.QUEUED if rank else T.TILED,
                            order=2, seed=rank + 1, y_begin=y_begin, y_end=y_end)
            return {k: torch.from_numpy(v) for k, v in out.items()}

        full = shard.search_row_band(torch.from_numpy(pp), times, vel, 3, 2, search=emulated_search)
        ref = oracle.search(pp, times, vel, 3, 2)
        for k in ref:
            a, b = full[k].numpy(), ref[k]
            assert a.shape == b.shape and ((a == b) | (np.isnan(a) & np.isnan(b))).all(), k
        # S2 sharded by image + one all-gather: bit-identical to a single-rank build (emulated kernel)
        from tests import emulated_binding
        cfg = synth.config(2, N=5, H=40, W=68, n_sources=2)
        st = synth.make_stack(cfg)
        tens = lambda a: torch.from_numpy(np.ascontiguousarray(a))
        whole = emulated_binding.make_psi_phi(tens(st.sci), tens(st.var), tens(st.mask), st.psf)
        gathered = shard.make_psi_phi_sharded(tens(st.sci), tens(st.var), tens(st.mask), st.psf,
                                              make=emulated_binding.make_psi_phi)
        assert gathered.shape == whole.shape
        assert torch.equal(gathered.view(torch.int32), whole.view(torch.int32))
        assert shard.image_shares(5, world) == [(0, 3), (3, 5)]
        t = shard.max_over_ranks(10.0 + 5.0 * rank)
        n = shard.total_over_ranks(100.0 * (rank + 1))
        assert t == 10.0 + 5.0 * (world - 1) and n == 100.0 * world * (world + 1) / 2
        assert shard.rank_seed(3, rank) != shard.rank_seed(3, (rank + 1) % world)
        ret[rank] = "ok"
    finally:
        dist.destroy_process_group()


def test_row_bands_partition():
    for H, n in ((4096, 8), (23, 2), (5, 8), (1, 1), (100, 3)):
        b = shard.row_bands(H, n)
        assert len(b) == n and b[0][0] == 0 and b[-1][1] == H
        assert all(b[i][1] == b[i + 1][0] for i in range(n - 1))
        sizes = [y1 - y0 for y0, y1 in b]
        assert max(sizes) - min(sizes) <= 1


def test_single_process_degrades():
    assert shard.world() == (0, 1)
    assert shard.max_over_ranks(3.5) == 3.5 and shard.total_over_ranks(7.0) == 7.0


def test_world_size_2_gloo(orc):
    ctx = mp.get_context("spawn")
    ret = ctx.Manager().dict()
    port = _free_port()
    from tests import simt_build
    simt_build.load("tiled_simt")            # compile once, before the ranks race for it
    simt_build.build_abi_lib()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, ret)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(180)
    assert all(p.exitcode == 0 for p in procs), [p.exitcode for p in procs]
    assert dict(ret) == {0: "ok", 1: "ok"}
