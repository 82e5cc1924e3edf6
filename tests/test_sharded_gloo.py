"""world_size-2 gloo test (CPU) of the band-sharded driver (paper_2607_03226_b200/sharded.py, PAPER.md:115-121
Eq. 14): band split, the buffer of a rank's terms, the one all-reduce per iteration, the outer loop.  The local engine is a
CPU stand-in built on the oracle (this is a test: tests may use oracle/), so the arithmetic checked here is: the terms of
the shards add up to the unsharded update, on every rank, with the same iteration count."""
import os
import socket

import numpy as np
import torch
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


class OracleShard:
    """The four methods ShardedSolver needs, on the CPU oracle: a shard's terms of (theta_SI, theta_en, q) are its own
    moments rescaled from the shard's normalisation (beta_r, sum C_r) to the whole table's."""

    def __init__(self, sub, whole):
        from oracle.ref import RefSolver
        Cw, tw = np.asarray(whole["bands"]["C"]), np.asarray(whole["bands"]["tau"])
        Cs, ts = np.asarray(sub["bands"]["C"]), np.asarray(sub["bands"]["tau"])
        self.fb, self.fc = (Cs / ts).sum() / (Cw / tw).sum(), Cs.sum() / Cw.sum()
        self.T_ref = whole["T_ref"]
        self.r = RefSolver(sub, share=Cs / Cw.sum())

    def sweep(self):
        self.r.sweep()

    def update_temperature(self, sync=False):
        self.T_old = self.r.get_T(0)  # the iterate the update starts from (the oracle's own update overwrites it)
        return self.r.update_temperature()

    def export_moments(self):
        th_SI = (self.r.get_T(2) - self.T_ref) * self.fb
        th_en = (self.r.get_T(1) - self.T_ref) * self.fc
        return torch.from_numpy(np.concatenate([th_SI, th_en, self.r.get_q().ravel()]))

    def import_moments(self, buf):
        n = self.r.n_cells
        T_old = self.T_old
        T_new = self.T_ref + buf[:n].numpy()
        self.r.set_T(T_new)
        self.last = buf.numpy().copy()
        return float(np.abs(T_new - T_old).max())

    def close(self):
        self.r.close()


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from oracle.ref import RefSolver
    from paper_2607_03226_b200 import replicas, sharded
    from paper_2607_03226_b200 import workloads as wl
    dist = replicas.init("gloo")
    pr = wl.config_nongray_square(n=12, B=5, D=8)
    s = sharded.ShardedSolver(pr, rank, world, dist=dist, make_solver=lambda sub, whole: OracleShard(sub, whole))
    ref = RefSolver(pr)
    worst = 0.0
    for _ in range(3):
        dT, _ = s.step("plain")
        ref.sweep()
        dr = ref.update_temperature()
        n = ref.n_cells
        worst = max(worst, np.abs(s.local.last[:n] - (ref.get_T(2) - pr["T_ref"])).max() / np.abs(ref.get_T(2) - pr["T_ref"]).max(),
                    np.abs(s.local.last[n:2 * n] - (ref.get_T(1) - pr["T_ref"])).max() / np.abs(ref.get_T(1) - pr["T_ref"]).max(),
                    np.abs(s.local.last[2 * n:] - ref.get_q().ravel()).max() / np.abs(ref.get_q()).max(), abs(dT - dr) / dr)
    res = s.solve(1e-9, 2000, "plain")
    rr = RefSolver(pr).solve(1e-9, 2000, "plain")
    out.put((rank, s.bands, worst, res["iters"], rr["iters"], float(s.local.r.get_T(0).sum())))
    replicas.barrier(dist)
    dist.destroy_process_group()


def test_two_band_shards_add_up_to_the_unsharded_update():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == [0, 2, 4] and res[1][1] == [1, 3]          # round-robin split
    for rank, bands, worst, it_sharded, it_ref, _ in res:
        assert worst <= 1e-10, worst                                  # the terms add up to the unsharded moments
        assert it_sharded + 3 == it_ref                               # solve() continued after the three steps above
    assert res[0][5] == res[1][5]                                     # the same field on both ranks, bit for bit


def test_shard_bands_partition():
    from paper_2607_03226_b200.sharded import shard_bands
    for B, world in ((30, 4), (7, 7), (10, 3)):
        got = sorted(b for r in range(world) for b in shard_bands(B, r, world))
        assert got == list(range(B))
    import pytest
    with pytest.raises(ValueError):
        shard_bands(3, 0, 4)
