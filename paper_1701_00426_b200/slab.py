"""Slab decomposition along x3: one process per GPU, one x3 slab per process.

The paper's code is single-device; its multi-device version is future work.
SURVEY.md section 8(e) gives the natural sharding of THIS path, built here (NEXT-2):

  * rank r of P owns the L3 = N3/P time slices x3 in [r*L3, (r+1)*L3) of both parities and holds
    them as an ordinary lattice of extents (N0, N1, N2, L3+2): local slice 0 and L3+1 are ghost copies
    of the neighbours' boundary slices (links: static, filled once; vectors: exchanged before every
    Dslash).  Ghost depth 1 makes the local x3 = global x3 - r*L3 + 1, so the LOCAL parity of a site is
    the opposite of its global parity (r*L3 is even because L3 is);
  * the staggered phases eta_mu do not depend on x3 (eta_3 = (-1)^(x0+x1+x2)) and the antiperiodic sign
    of the fermion field is applied to the halo data that crosses the global x3 boundary, so the slab's
    context has antiperiodic_t = 0 and needs no special kernel: only lqcd_dslash_slices (owned slices);
  * per Dslash: the two boundary slices of the input vector go to the +-x3 neighbours (N0*N1*N2/2 sites
    x 48 B = 786 kB per face at 32^4 fp64); the interior slices are computed while the halo is in
    flight, the two boundary slices after it arrived;
  * per CG iteration two all-reduces of one double (<p,q>, <r,r>), through the hooks of lqcd_set_slab.

Two transports:
  * "peer" (the native one, lqcd_peer_* in lqcd.h): faces and partial sums move through peer-to-peer device
    memory inside the library's own kernels -- no Python, no communication library and no host code between the
    kernels of a solve; this module only creates the per-rank blocks and hands every rank the others' addresses
    (CUDA IPC handles gathered with torch.distributed for one process per GPU; plain pointers for ranks that
    share a process);
  * "hooks" (lqcd_set_slab): the library calls back into this module for every halo exchange and all-reduce
    (SlabComm: torch.distributed, NCCL on GPUs, gloo in the CPU tests) -- the portable fallback.

Everything here is plumbing: index bookkeeping in numpy (SlabGeometry, covered by CPU tests), the
exchange through torch.distributed (SlabComm: NCCL on GPUs, gloo in the CPU tests), and argument
marshalling (SlabLattice).  Every arithmetic step runs in the CUDA kernels of liblqcd_b200.so.
"""
from __future__ import annotations

import ctypes as C

import numpy as np


class SlabGeometry:
    """Host-side bookkeeping of one rank's slab.  numpy only; no GPU, no torch."""

    def __init__(self, dims, world, rank, antiperiodic_t=True):
        dims = tuple(int(d) for d in dims)
        if len(dims) != 4 or any(d < 2 or d % 2 for d in dims):
            raise ValueError("dims must be four even extents >= 2")
        if world < 1 or not (0 <= rank < world):
            raise ValueError(f"bad rank {rank} of {world}")
        if dims[3] % world or (dims[3] // world) % 2:
            raise ValueError(f"N3 = {dims[3]} must split into {world} slabs of even thickness")
        self.dims, self.world, self.rank = dims, world, rank
        self.L3 = dims[3] // world
        self.local_dims = (dims[0], dims[1], dims[2], self.L3 + 2)
        self.x3_lo, self.x3_hi = 1, self.L3 + 1          # owned local slices [x3_lo, x3_hi)
        self.up, self.down = (rank + 1) % world, (rank - 1) % world
        # sign applied by the SENDER to a boundary slice whose hop crosses the global x3 boundary
        # (reading R4: s+ = -1 at x3 = N3-1, s- = -1 at x3 = 0)
        ap = -1.0 if antiperiodic_t else 1.0
        self.sign_send_up = ap if rank == world - 1 else 1.0      # my top slice -> up's bottom ghost
        self.sign_send_down = ap if rank == 0 else 1.0            # my bottom slice -> down's top ghost
        self.slice_sites = dims[0] * dims[1] * dims[2]            # full-lattice sites per x3 slice
        self.V_local = self.slice_sites * (self.L3 + 2)

    def local_parity(self, global_parity: int) -> int:
        """Ghost depth 1 and an even slab offset: local parity = 1 - global parity."""
        return 1 - int(global_parity)

    def global_x3_of_local(self):
        """Global x3 of the local slices 0 .. L3+1 (periodic wrap)."""
        return [(self.rank * self.L3 - 1 + k) % self.dims[3] for k in range(self.L3 + 2)]

    def extract_full(self, field):
        """Full-lattice canonical array [V, ...] (lex order, x3 slowest) -> the slab's [V_local, ...]
        including both ghost slices (true neighbour values, NO boundary sign)."""
        f = np.asarray(field)
        s = self.slice_sites
        assert f.shape[0] == s * self.dims[3]
        return np.concatenate([f[g * s:(g + 1) * s] for g in self.global_x3_of_local()], axis=0)

    def half_index(self, dims, parity):
        """lex indices of the sites of `parity` in idxh order (same convention as lqcd_inputs)."""
        n0, n1, n2, n3 = dims
        lex = np.arange(n0 * n1 * n2 * n3)
        x0 = lex % n0
        x1 = (lex // n0) % n1
        x2 = (lex // (n0 * n1)) % n2
        x3 = lex // (n0 * n1 * n2)
        return lex[(x0 + x1 + x2 + x3) % 2 == parity]

    def extract_half(self, phi, global_parity):
        """Global half vector [V/2, 3] of `global_parity` -> local half vector of the opposite local
        parity [V_local/2, 3], ghosts included (unsigned)."""
        V = self.slice_sites * self.dims[3]
        full = np.zeros((V,) + phi.shape[1:], dtype=phi.dtype)
        full[self.half_index(self.dims, global_parity)] = phi
        return self.extract_full(full)[self.half_index(self.local_dims, self.local_parity(global_parity))]

    def insert_half(self, local_phi, global_parity, out):
        """Scatter the OWNED slices of a local half vector into the global half vector `out`."""
        lp = self.local_parity(global_parity)
        full_loc = np.zeros((self.V_local,) + local_phi.shape[1:], dtype=local_phi.dtype)
        full_loc[self.half_index(self.local_dims, lp)] = local_phi
        s = self.slice_sites
        V = s * self.dims[3]
        full = np.zeros((V,) + local_phi.shape[1:], dtype=local_phi.dtype)
        full[self.half_index(self.dims, global_parity)] = out
        gx3 = self.global_x3_of_local()
        for k in range(self.x3_lo, self.x3_hi):
            full[gx3[k] * s:(gx3[k] + 1) * s] = full_loc[k * s:(k + 1) * s]
        out[...] = full[self.half_index(self.dims, global_parity)]
        return out


class SlabComm:
    """Neighbour exchange and scalar all-reduce over torch.distributed (NCCL on GPUs; the CPU tests use
    gloo with CPU tensors).  world == 1 needs no process group: the slab is its own neighbour."""

    def __init__(self, world, rank):
        self.world, self.rank = int(world), int(rank)
        self.up, self.down = (rank + 1) % world, (rank - 1) % world

    def exchange_start(self, send_up, send_down, recv_from_down, recv_from_up):
        """Post: my top slice -> up's bottom ghost, my bottom slice -> down's top ghost.  Returns a
        handle for exchange_wait.  Tag 0 = data moving up, tag 1 = data moving down (with two ranks
        both messages go to the same peer)."""
        if self.world == 1:
            recv_from_down.copy_(send_up)
            recv_from_up.copy_(send_down)
            return []
        import torch.distributed as dist
        ops = [dist.P2POp(dist.isend, send_up, self.up, tag=0),
               dist.P2POp(dist.irecv, recv_from_down, self.down, tag=0),
               dist.P2POp(dist.isend, send_down, self.down, tag=1),
               dist.P2POp(dist.irecv, recv_from_up, self.up, tag=1)]
        return dist.batch_isend_irecv(ops)

    def exchange_wait(self, handle):
        for req in handle:
            req.wait()

    def allreduce_sum(self, tensor):
        if self.world > 1:
            import torch.distributed as dist
            dist.all_reduce(tensor, op=dist.ReduceOp.SUM)
        return tensor


class _RawDeviceDoubles:
    """Zero-copy view of `count` device doubles at a raw address (torch.as_tensor reads this)."""

    def __init__(self, ptr, count):
        self.__cuda_array_interface__ = {"shape": (int(count),), "typestr": "<f8", "data": (int(ptr), False),
                                         "version": 2}


class SlabLattice:
    """One rank's slab on one GPU: a Lattice of the local extents (ghost slices included), the halo
    buffers, and the hooks that let the library's solvers exchange halos and sum dot products through
    `comm` (a SlabComm, or any object with exchange_start / exchange_wait / allreduce_sum).
    Parities in this API are GLOBAL (the paper's even sites); the local flip is handled here."""

    def __init__(self, dims, world, rank, comm=None, prec=0, recon=0, antiperiodic_t=True, device=0, options=None,
                 transport="hooks"):
        from .binding import Lattice, HALO_FN, ALLREDUCE_FN
        if transport not in ("hooks", "peer"):
            raise ValueError("transport must be 'hooks' or 'peer'")
        self.transport = transport
        self.geo = SlabGeometry(dims, world, rank, antiperiodic_t)
        self.comm = comm if comm is not None else SlabComm(world, rank)
        self.lat = Lattice(self.geo.local_dims, prec=prec, recon=recon, antiperiodic_t=False, device=device,
                           options=options)
        self.torch = self.lat.torch
        self.hook_error = None
        if transport == "peer":
            g = self.geo
            self.peer_block = self.lat.peer_init(world, rank, g.x3_lo, g.x3_hi, g.local_parity(0),
                                                 g.sign_send_up, g.sign_send_down)
            if world == 1:
                self.lat.peer_connect([self.peer_block])
            return
        hb = self.lat.halo_bytes
        self._send_up, self._send_down, self._from_down, self._from_up = (self.lat._buf(hb) for _ in range(4))
        self._halo_cb = HALO_FN(self._halo_hook)
        self._allreduce_cb = ALLREDUCE_FN(self._allreduce_hook)
        self.lat.set_slab(self.geo.x3_lo, self.geo.x3_hi, self.geo.local_parity(0), self._halo_cb, self._allreduce_cb)

    def close(self):
        """Peer transport between processes: a neighbour's last kernel may still be storing into this rank's block
        (the faces K2 pushes after the final iteration have no reader), and freeing the block under it would fault the
        neighbour's GPU.  So every rank finishes its own stream and meets the others before anyone frees (lqcd.h,
        "Teardown").  Ranks that share a process (connect_local) are closed by one thread after all have finished."""
        if getattr(self, "_ipc_connected", False) and self.lat._ctx:
            import torch.distributed as dist
            self.lat.synchronize()
            if dist.is_initialized():
                dist.barrier()
            self._ipc_connected = False
        self.lat.close()

    # -- peer transport: hand every rank the other ranks' blocks ------------------------------------------
    @staticmethod
    def connect_local(slabs):
        """Ranks that share a process (one context each, e.g. the single-GPU validation harness): plain pointers."""
        blocks = [s.peer_block for s in sorted(slabs, key=lambda s: s.geo.rank)]
        for s in slabs:
            s.lat.peer_connect(blocks)

    def connect_ipc(self):
        """One process per GPU (torchrun): gather the CUDA IPC handles of all blocks with torch.distributed, map
        the other ranks' blocks, connect.  Collective over the default process group."""
        import torch.distributed as dist
        g = self.geo
        handles = [None] * g.world
        dist.all_gather_object(handles, self.lat.peer_export())
        blocks = [self.peer_block if r == g.rank else self.lat.peer_import(r, handles[r]) for r in range(g.world)]
        self.lat.peer_connect(blocks)
        self._ipc_connected = True
        dist.barrier()

    def set_lockstep(self, barrier):
        """Validation on ONE GPU: after every launch that publishes to the peers, finish this rank's stream and
        meet the other ranks (host threads) at `barrier` -- no kernel ever waits for another rank's kernel."""
        from .binding import PHASE_FN

        def phase(user, what):
            try:
                self.lat.synchronize()
                barrier.wait()
                return 0
            except Exception as e:        # an exception must not unwind through the C frames
                self.hook_error = e
                return 1
        self.lat.set_phase_hook(PHASE_FN(phase) if barrier is not None else None)

    # -- fields ------------------------------------------------------------------------------
    def pack_links(self, U_global):
        """Global canonical links [V][4][3][3] -> this rank's native link field (ghost slices included:
        the backward x3 hop of the first owned slice reads U_3 of the slice below)."""
        return self.lat.pack_links(np.ascontiguousarray(self.geo.extract_full(U_global)))

    def pack_backfield(self, theta_global):
        """Global phases theta[V][4] -> this rank's native backfield (ghost slices included, like the links: the
        backward x3 hop of the first owned slice carries the phase of the link in the slice below).  Attach it with
        self.lat.set_backfield(...); both transports."""
        return self.lat.pack_backfield(np.ascontiguousarray(self.geo.extract_full(theta_global)))

    def pack_spinor(self, phi_global, global_parity):
        """Global half vector -> native local vector; the ghost slices start out ZERO (they are
        filled by the halo exchange, never by the host)."""
        g = self.geo
        loc = g.extract_half(phi_global, global_parity)
        s3 = g.slice_sites // 2
        loc[:s3] = 0
        loc[-s3:] = 0
        return self.lat.pack_spinor(np.ascontiguousarray(loc), g.local_parity(global_parity))

    def unpack_spinor(self, native, global_parity, out_global):
        """Owned slices of a native local vector -> their place in the global half vector."""
        loc = self.lat.unpack_spinor(native, self.geo.local_parity(global_parity))
        return self.geo.insert_half(loc, global_parity, out_global)

    def new_spinor(self):
        t = self.lat.new_spinor()
        t.zero_()
        return t

    # -- hooks called from inside liblqcd_b200.so (lqcd_set_slab) ---------------------------------
    # The library's kernels run on the stream captured when the Lattice was created; torch copies and
    # collectives run on torch's CURRENT stream.  Every piece of communication is therefore issued under
    # `with torch.cuda.stream(lat.stream)`, so that it stays ordered with the kernels even when the caller
    # has entered another stream context.
    def _halo_start(self, vec_ptr):
        g, lat = self.geo, self.lat
        lat.halo_pack_faces(self._send_up, self._send_down, vec_ptr, g.sign_send_up, g.sign_send_down)
        with self.torch.cuda.stream(lat.stream):
            return self.comm.exchange_start(self._send_up, self._send_down, self._from_down, self._from_up)

    def _halo_finish(self, vec_ptr, handle):
        g, lat = self.geo, self.lat
        with self.torch.cuda.stream(lat.stream):
            self.comm.exchange_wait(handle)
        lat.halo_unpack_ghosts(vec_ptr, self._from_down, self._from_up)

    def _halo_hook(self, user, vec_ptr, parity):
        try:
            self._halo_finish(vec_ptr, self._halo_start(vec_ptr))
            return 0
        except Exception as e:  # an exception must not unwind through the C frames
            self.hook_error = e
            return 1

    def _allreduce_hook(self, user, dev_ptr, count):
        try:
            with self.torch.cuda.stream(self.lat.stream):
                t = self.torch.as_tensor(_RawDeviceDoubles(dev_ptr, count), device=self.lat.device)
                self.comm.allreduce_sum(t)
            return 0
        except Exception as e:
            self.hook_error = e
            return 1

    # -- the hot path -----------------------------------------------------------------------------
    def dslash(self, out_global_parity, out, inp, links, overlap=True):
        """out = D inp on the owned slices; halo of `inp` exchanged first.  With overlap, the interior
        slices are computed while the two faces are in flight, the boundary slices afterwards."""
        g, lat = self.geo, self.lat
        lp = g.local_parity(out_global_parity)
        if self.transport == "peer":          # the library pushes the faces and the kernel waits for them
            lat.dslash(lp, out, inp, links)
            self._raise_hook_error()
            return
        handle = self._halo_start(inp.data_ptr())
        lo, hi = g.x3_lo, g.x3_hi
        if overlap and hi - lo > 2:
            lat.dslash_slices(lp, out, inp, links, lo + 1, hi - 1)
            self._halo_finish(inp.data_ptr(), handle)
            lat.dslash_slices(lp, out, inp, links, lo, lo + 1)
            lat.dslash_slices(lp, out, inp, links, hi - 1, hi)
        else:
            self._halo_finish(inp.data_ptr(), handle)
            lat.dslash_slices(lp, out, inp, links, lo, hi)

    def fermion_force(self, xs, links, coeffs):
        """lqcd_fermion_force on the slab (both transports): xs = the solutions on the paper's even sites (native local
        vectors; their ghost slices are overwritten by the halo exchange).  Returns the native (tamat) force field of
        the LOCAL lattice; only the owned links are written -- collect them with unpack_tamat_owned."""
        try:
            return self.lat.fermion_force(xs, links, coeffs)
        finally:
            self._raise_hook_error()

    def unpack_tamat_owned(self, native, out_global):
        """Owned links of a native local tamat field (the fermion force) -> their place in the global canonical field
        out_global[V][4][3][3]."""
        loc = self.lat.unpack_tamat(native)
        g = self.geo
        s = g.slice_sites
        gx3 = g.global_x3_of_local()
        for k in range(g.x3_lo, g.x3_hi):
            out_global[gx3[k] * s:(gx3[k] + 1) * s] = loc[k * s:(k + 1) * s]
        return out_global

    def _raise_hook_error(self):
        if self.hook_error is not None:
            e, self.hook_error = self.hook_error, None
            raise e

    def mdagm(self, out_e, in_e, links, mass, sigma=0.0):
        self.lat.mdagm(out_e, in_e, links, mass, sigma)
        self._raise_hook_error()

    def cg_multishift(self, xs, b_e, links, mass, shifts, tol, max_iter, raise_on_max_iter=True):
        """Vectors live on the paper's (global) even sites.  Same call as Lattice.cg_multishift; the
        library calls back into the halo / all-reduce hooks every iteration."""
        try:
            return self.lat.cg_multishift(xs, b_e, links, mass, shifts, tol, max_iter, raise_on_max_iter)
        finally:
            self._raise_hook_error()

    def rational_apply(self, y_e, b_e, links, mass, shifts, c0, coeffs, tol, max_iter, raise_on_max_iter=True):
        try:
            return self.lat.rational_apply(y_e, b_e, links, mass, shifts, c0, coeffs, tol, max_iter, raise_on_max_iter)
        finally:
            self._raise_hook_error()
