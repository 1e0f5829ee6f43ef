"""-m "not gpu": host logic of the x3-slab decomposition (paper_1701_00426_b200/slab.py, NEXT-2).

The design claim -- a slab with one ghost slice per side is an ORDINARY lattice with antiperiodic_t = 0,
the opposite local parity, and the boundary sign carried by the halo data -- is checked against the
oracle on the CPU: the oracle applied to each rank's local fields reproduces, on the owned slices, the
oracle applied to the global lattice.  The exchange itself runs under gloo with world_size 2."""
import os
import subprocess
import sys

import numpy as np
import pytest

import lqcd_inputs as gen
import oracle
from paper_1701_00426_b200.slab import SlabGeometry

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def signed_local_half(geo, phi, gp, ap):
    """What a rank's local vector holds after a halo exchange: true neighbour slices, with the sender's
    boundary sign on the ghosts."""
    loc = geo.extract_half(phi, gp)
    s3 = geo.slice_sites // 2
    # bottom ghost came from `down`'s top slice (sender sign_send_up of that rank); top ghost from `up`
    down = SlabGeometry(geo.dims, geo.world, geo.down, ap)
    up = SlabGeometry(geo.dims, geo.world, geo.up, ap)
    loc[:s3] *= down.sign_send_up
    loc[-s3:] *= up.sign_send_down
    return loc


@pytest.mark.parametrize("ap", [True, False])
@pytest.mark.parametrize("world", [1, 2, 4])
def test_slab_is_an_ordinary_lattice_with_signed_ghosts(world, ap):
    dims = (4, 6, 2, 8)
    rng = np.random.default_rng(21)
    U = gen.haar_like_links(dims, rng)
    psi = gen.gaussian_spinor(dims, rng)
    for gp_out in (0, 1):
        phi_in = oracle.full_to_half(dims, 1 - gp_out, psi)
        want = oracle.dslash_half(dims, U, gp_out, phi_in, antiperiodic_t=ap)
        got = np.zeros_like(want)
        for rank in range(world):
            geo = SlabGeometry(dims, world, rank, ap)
            assert geo.local_parity(gp_out) == 1 - gp_out
            U_loc = np.ascontiguousarray(geo.extract_full(U))
            in_loc = signed_local_half(geo, phi_in, 1 - gp_out, ap)
            out_loc = oracle.dslash_half(geo.local_dims, U_loc, geo.local_parity(gp_out), in_loc,
                                         antiperiodic_t=False)
            geo.insert_half(out_loc, gp_out, got)
        assert rel(got, want) < 1e-14, (world, ap, gp_out)


def test_geometry_roundtrip_and_errors():
    dims = (4, 4, 2, 8)
    phi = gen.gaussian_half_spinor(dims, 3)
    out = np.zeros_like(phi)
    for rank in range(2):
        geo = SlabGeometry(dims, 2, rank)
        assert geo.local_dims == (4, 4, 2, 6) and (geo.x3_lo, geo.x3_hi) == (1, 5)
        geo.insert_half(geo.extract_half(phi, 0), 0, out)
    assert np.array_equal(out, phi)
    g0, g1 = SlabGeometry(dims, 2, 0), SlabGeometry(dims, 2, 1)
    assert g0.global_x3_of_local() == [7, 0, 1, 2, 3, 4] and g1.global_x3_of_local() == [3, 4, 5, 6, 7, 0]
    assert (g0.sign_send_down, g0.sign_send_up, g1.sign_send_down, g1.sign_send_up) == (-1.0, 1.0, 1.0, -1.0)
    assert SlabGeometry(dims, 1, 0).sign_send_up == -1.0 and SlabGeometry(dims, 1, 0, False).sign_send_up == 1.0
    with pytest.raises(ValueError):
        SlabGeometry(dims, 8, 0)        # slabs of thickness 1
    with pytest.raises(ValueError):
        SlabGeometry(dims, 3, 0)
    with pytest.raises(ValueError):
        SlabGeometry(dims, 2, 2)


_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import numpy as np, torch
import torch.distributed as dist
import lqcd_inputs as gen
from paper_1701_00426_b200.slab import SlabGeometry, SlabComm
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
dims = (4, 4, 2, 8)
phi = gen.gaussian_half_spinor(dims, 7)              # same global vector on both ranks
geo = SlabGeometry(dims, world, rank)
comm = SlabComm(world, rank)
loc = geo.extract_half(phi, 0)                        # ghosts hold the TRUE neighbour values
s3 = geo.slice_sites // 2
top = torch.from_numpy(np.ascontiguousarray(loc[-2 * s3:-s3]) * geo.sign_send_up)
bot = torch.from_numpy(np.ascontiguousarray(loc[s3:2 * s3]) * geo.sign_send_down)
from_down, from_up = torch.empty_like(top), torch.empty_like(top)
comm.exchange_wait(comm.exchange_start(top, bot, from_down, from_up))
sign_b = -1.0 if rank == 0 else 1.0                   # my bottom ghost crossed the global boundary
sign_t = -1.0 if rank == world - 1 else 1.0
assert np.array_equal(from_down.numpy(), sign_b * loc[:s3]), "bottom ghost"
assert np.array_equal(from_up.numpy(), sign_t * loc[-s3:]), "top ghost"
t = torch.tensor([1.5 + rank, -2.0], dtype=torch.float64)
comm.allreduce_sum(t)
assert t.tolist() == [4.0, -4.0], t
dist.barrier()
dist.destroy_process_group()
print("rank", rank, "ok")
"""


def test_slab_exchange_gloo_world2(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(_WORKER % ROOT)
    port = 29950 + os.getpid() % 40
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, o
        assert f"rank {r} ok" in o


_WORKER_IPC = r"""
import os, sys
sys.path.insert(0, %r)
import torch.distributed as dist
from paper_1701_00426_b200.slab import SlabLattice, SlabGeometry
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)


class FakeLat:                      # stands for the Lattice of a GPU box: records what the plumbing hands to the library
    def __init__(self):
        self.connected = None
        self.events = []
    def peer_export(self):
        return bytes([rank]) * 64   # this rank's "IPC handle"
    def peer_import(self, r, handle):
        assert handle == bytes([r]) * 64, (r, handle)
        return 1000 + r             # "device address" of rank r's block mapped into this process
    def peer_connect(self, blocks):
        self.connected = list(blocks)
    _ctx = 1
    def synchronize(self):
        self.events.append("sync")
    def close(self):
        self.events.append("close")
        self._ctx = None


sl = SlabLattice.__new__(SlabLattice)        # no GPU here: only the connect_ipc plumbing is under test
sl.geo = SlabGeometry((4, 4, 2, 8), world, rank)
sl.lat = FakeLat()
sl.peer_block = 7000 + rank
sl.connect_ipc()
want = [7000 + rank if r == rank else 1000 + r for r in range(world)]
assert sl.lat.connected == want, (sl.lat.connected, want)
# teardown: close() finishes the rank's stream, then meets the other ranks, then frees -- rank 1 arrives 1.5 s late and
# rank 0 must not have freed its block before
import time
if rank == 1:
    time.sleep(1.5)
t0 = time.time()
sl.close()
waited = time.time() - t0
assert sl.lat.events == ["sync", "close"], sl.lat.events
assert rank == 1 or waited > 1.0, waited
dist.destroy_process_group()
print("rank", rank, "ok")
"""


def test_peer_connect_ipc_plumbing_gloo_world2(tmp_path):
    """SlabLattice.connect_ipc (the one-process-per-GPU set-up of the peer transport) under gloo with two CPU
    processes and a stand-in for the GPU context: every rank gathers all handles, maps the OTHER ranks' blocks, keeps
    its own, and connects with the blocks in rank order; close() synchronises, waits for the other ranks, then frees."""
    script = tmp_path / "w_ipc.py"
    script.write_text(_WORKER_IPC % ROOT)
    port = 29870 + os.getpid() % 40
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, o
        assert f"rank {r} ok" in o
