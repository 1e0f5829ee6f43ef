"""ctypes binding of include/lqcd.h -- same names, argument marshalling only.

`lib` is the raw ctypes handle (lib.lqcd_dslash(...) etc. with C signatures).  `Lattice` is a
small convenience wrapper that owns a context plus the torch tensors used as device memory; it
does no arithmetic.
"""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
lib_path = os.path.join(HERE, "liblqcd_b200.so")

OK, ERR_ARG, ERR_UNSUPPORTED, ERR_CUDA, ERR_NOT_CONVERGED, ERR_WORKSPACE = range(6)
F64, F32 = 0, 1
RECON_18, RECON_12 = 0, 1
EVEN, ODD = 0, 1
MAX_SHIFTS = 32
NOALLOC_SCRATCH_BYTES = 8 << 20   # LQCD_NOALLOC_SCRATCH_BYTES


class LqcdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"lqcd error {code}: {msg}")
        self.code = code


def _load():
    if not os.path.exists(lib_path):
        raise ImportError(
            f"{lib_path} is missing: build it with `python paper_1701_00426_b200/build.py` "
            "(or __graft_entry__.build()).  There is no fallback path.")
    return C.CDLL(lib_path)


lib = _load()

_vp, _i, _d, _sz = C.c_void_p, C.c_int, C.c_double, C.c_size_t
_pi, _pd = C.POINTER(C.c_int), C.POINTER(C.c_double)
HALO_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_int)        # lqcd_halo_fn
ALLREDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_int)   # lqcd_allreduce_fn
PHASE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int)                   # lqcd_phase_fn
_sig = {
    "lqcd_version": (C.c_char_p, []),
    "lqcd_create": (_i, [C.POINTER(_vp), C.POINTER(_i), _i, _i, _i, _i, _vp]),
    "lqcd_destroy": (_i, [_vp]),
    "lqcd_last_error": (C.c_char_p, [_vp]),
    "lqcd_set_option": (_i, [_vp, C.c_char_p, C.c_long]),
    "lqcd_get_option": (C.c_long, [_vp, C.c_char_p]),
    "lqcd_spinor_bytes": (_sz, [_vp]),
    "lqcd_links_bytes": (_sz, [_vp]),
    "lqcd_workspace_bytes": (_sz, [_vp, _i]),
    "lqcd_set_workspace": (_i, [_vp, _vp, _sz]),
    "lqcd_pack_links": (_i, [_vp, _vp, _vp]),
    "lqcd_pack_spinor": (_i, [_vp, _i, _vp, _vp]),
    "lqcd_unpack_spinor": (_i, [_vp, _i, _vp, _vp]),
    "lqcd_dslash": (_i, [_vp, _i, _vp, _vp, _vp]),
    "lqcd_dslash_multi": (_i, [_vp, _i, _i, C.POINTER(_vp), C.POINTER(_vp), _vp]),
    "lqcd_backfield_bytes": (_sz, [_vp]),
    "lqcd_pack_backfield": (_i, [_vp, _vp, _vp]),
    "lqcd_set_backfield": (_i, [_vp, _vp]),
    "lqcd_dslash_backfield": (_i, [_vp, _i, _vp, _vp, _vp, _vp]),
    "lqcd_mdagm": (_i, [_vp, _vp, _vp, _vp, _d, _d]),
    "lqcd_mdagm_noalloc": (_i, [_vp, _vp, _vp, _vp, _d, _d]),
    "lqcd_cg": (_i, [_vp, _vp, _vp, _vp, _d, _d, _i, _pi, _pd]),
    "lqcd_cg_multishift": (_i, [_vp, _i, _pd, _vp, C.POINTER(_vp), _vp, _d, _d, _i, _pi, _pi, _pd]),
    "lqcd_rational_apply": (_i, [_vp, _i, _pd, _d, _pd, _vp, _vp, _vp, _d, _d, _i, _pi, _pi]),
    "lqcd_force_bytes": (_sz, [_vp]),
    "lqcd_tamat_bytes": (_sz, [_vp]),
    "lqcd_unpack_tamat": (_i, [_vp, _vp, _vp]),
    "lqcd_fermion_force": (_i, [_vp, _i, _pd, C.POINTER(_vp), _vp, _vp]),
    "lqcd_unpack_force": (_i, [_vp, _vp, _vp]),
    "lqcd_staples_workspace_bytes": (_sz, [_vp]),
    "lqcd_gauge_staples": (_i, [_vp, _vp, _vp, _d, _d]),
    "lqcd_dslash_slices": (_i, [_vp, _i, _vp, _vp, _vp, _i, _i]),
    "lqcd_halo_bytes": (_sz, [_vp]),
    "lqcd_halo_pack": (_i, [_vp, _vp, _vp, _i, _d]),
    "lqcd_halo_unpack": (_i, [_vp, _vp, _vp, _i]),
    "lqcd_halo_pack_faces": (_i, [_vp, _vp, _vp, _vp, _d, _d]),
    "lqcd_halo_unpack_ghosts": (_i, [_vp, _vp, _vp, _vp]),
    "lqcd_set_slab": (_i, [_vp, _i, _i, _i, HALO_FN, ALLREDUCE_FN, _vp]),
    "lqcd_peer_block_bytes": (_sz, [_vp]),
    "lqcd_peer_init": (_i, [_vp, _i, _i, _i, _i, _i, _d, _d, C.POINTER(_vp)]),
    "lqcd_peer_export": (_i, [_vp, _vp]),
    "lqcd_peer_import": (_i, [_vp, _i, _vp, C.POINTER(_vp)]),
    "lqcd_peer_connect": (_i, [_vp, C.POINTER(_vp)]),
    "lqcd_peer_disconnect": (_i, [_vp]),
    "lqcd_set_phase_hook": (_i, [_vp, PHASE_FN, _vp]),
    "lqcd_peer_selftest": (_i, [_vp, _i, _i, _i, _pi]),
    "lqcd_solver_history": (_i, [_vp, _i, _pd, _pd, _pd]),
    "lqcd_dslash_host": (_i, [_vp, _i, _vp, _vp, _vp]),
    "lqcd_dslash_host_vectors": (_i, [_vp, _i, _vp, _vp, _vp]),
    "lqcd_cg_multishift_host": (_i, [_vp, _i, _pd, _vp, _vp, _vp, _d, _d, _i, _pi, _pi, _pd]),
    "lqcd_dslash_host_vectors_batch": (_i, [_vp, _i, _pi, C.POINTER(_vp), C.POINTER(_vp), _vp]),
    "lqcd_cg_multishift_host_vectors": (_i, [_vp, _i, _pd, _vp, _vp, _vp, _d, _d, _i, _pi, _pi, _pd]),
    "lqcd_measure_fp64_peak": (_i, [_vp, _pd]),
    "lqcd_measure_hbm_read": (_i, [_vp, _vp, _sz, _pd]),
}
for _name, (_res, _args) in _sig.items():
    _f = getattr(lib, _name)
    _f.restype = _res
    _f.argtypes = _args


def version() -> str:
    return lib.lqcd_version().decode()


class Lattice:
    """One lqcd context plus torch tensors as device memory.  Marshalling only.

    All numpy arguments / results are complex128 arrays in the canonical layout
    (include/lqcd.h).  Native device buffers are opaque uint8 torch tensors.
    """

    def __init__(self, dims, prec=F64, recon=RECON_18, antiperiodic_t=True, device=0, options=None):
        import torch  # device memory and streams only

        if not torch.cuda.is_available():
            raise LqcdError(ERR_CUDA, "no CUDA device: the lqcd_b200 path has no CPU fallback")
        self.torch = torch
        self.dims = tuple(int(d) for d in dims)
        self.prec, self.recon = prec, recon
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.stream = torch.cuda.current_stream(self.device)
        self._ctx = _vp()
        rc = lib.lqcd_create(C.byref(self._ctx), (C.c_int * 4)(*self.dims), prec, recon,
                             int(bool(antiperiodic_t)), device, _vp(self.stream.cuda_stream))
        if rc:
            raise LqcdError(rc, lib.lqcd_last_error(None).decode())
        for k, v in (options or {}).items():
            self.set_option(k, v)
        self.V = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        self.Vh = self.V // 2
        self._ws = None
        self._ws_shifts = 0

    # -- plumbing ------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_ctx", None):
            lib.lqcd_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, allow=()):
        if rc and rc not in allow:
            raise LqcdError(rc, lib.lqcd_last_error(self._ctx).decode())
        return rc

    def set_option(self, name, value):
        self._check(lib.lqcd_set_option(self._ctx, name.encode(), int(value)))

    def get_option(self, name):
        return int(lib.lqcd_get_option(self._ctx, name.encode()))

    @property
    def launches(self):
        return self.get_option("launches")

    @property
    def spinor_bytes(self):
        return int(lib.lqcd_spinor_bytes(self._ctx))

    @property
    def links_bytes(self):
        return int(lib.lqcd_links_bytes(self._ctx))

    def _buf(self, nbytes):
        return self.torch.empty(nbytes, dtype=self.torch.uint8, device=self.device)

    def new_spinor(self):
        return self._buf(self.spinor_bytes)

    def ensure_workspace(self, nshift=1, min_bytes=0):
        need = max(int(lib.lqcd_workspace_bytes(self._ctx, nshift)), int(min_bytes))
        if self._ws is None or need > self._ws.numel():
            self._ws = self._buf(need)
            self._check(lib.lqcd_set_workspace(self._ctx, _vp(self._ws.data_ptr()), self._ws.numel()))

    def synchronize(self):
        self.stream.synchronize()

    # -- canonical <-> native ----------------------------------------------------------------
    def _to_dev(self, arr):
        import numpy as np
        a = np.ascontiguousarray(arr, dtype=np.complex128)
        with self.torch.cuda.stream(self.stream):      # the upload is ordered with the context's kernels
            return self.torch.from_numpy(a.view(np.float64).reshape(-1)).to(self.device)

    def pack_links(self, U):
        """U: complex128 [V][4][3][3] (numpy) -> native device buffer."""
        assert U.shape == (self.V, 4, 3, 3)
        canon = self._to_dev(U)
        native = self._buf(self.links_bytes)
        self._check(lib.lqcd_pack_links(self._ctx, _vp(native.data_ptr()), _vp(canon.data_ptr())))
        self.synchronize()
        return native

    def pack_spinor(self, phi, parity):
        assert phi.shape == (self.Vh, 3)
        canon = self._to_dev(phi)
        native = self.new_spinor()
        self._check(lib.lqcd_pack_spinor(self._ctx, parity, _vp(native.data_ptr()), _vp(canon.data_ptr())))
        self.synchronize()
        return native

    def unpack_spinor(self, native, parity):
        import numpy as np
        canon = self.torch.empty(self.Vh * 6, dtype=self.torch.float64, device=self.device)
        self._check(lib.lqcd_unpack_spinor(self._ctx, parity, _vp(canon.data_ptr()), _vp(native.data_ptr())))
        self.synchronize()
        return canon.cpu().numpy().view(np.complex128).reshape(self.Vh, 3)

    # -- the hot path (async unless stated) ---------------------------------------------------
    def dslash(self, parity, out, inp, links):
        self._check(lib.lqcd_dslash(self._ctx, parity, _vp(out.data_ptr()), _vp(inp.data_ptr()), _vp(links.data_ptr())))

    def dslash_multi(self, parity, outs, inps, links):
        """block Dslash: outs[r] = D inps[r]; every link loaded once per block of right-hand sides.  async."""
        n = len(outs)
        assert len(inps) == n
        po = (_vp * n)(*[o.data_ptr() for o in outs])
        pi = (_vp * n)(*[i.data_ptr() for i in inps])
        self._check(lib.lqcd_dslash_multi(self._ctx, parity, n, po, pi, _vp(links.data_ptr())))

    def pack_backfield(self, theta):
        """theta: float64 [V][4] (numpy), the per-link U(1) phases -> native device buffer."""
        import numpy as np
        assert theta.shape == (self.V, 4)
        a = np.ascontiguousarray(theta, dtype=np.float64)
        with self.torch.cuda.stream(self.stream):
            canon = self.torch.from_numpy(a.reshape(-1)).to(self.device)
        native = self._buf(int(lib.lqcd_backfield_bytes(self._ctx)))
        self._check(lib.lqcd_pack_backfield(self._ctx, _vp(native.data_ptr()), _vp(canon.data_ptr())))
        self.synchronize()
        return native

    def set_backfield(self, native=None):
        """attach a native phase field to every later Dslash of this context (None detaches)."""
        self._backfield = native            # keeps the buffer alive while attached
        self._check(lib.lqcd_set_backfield(self._ctx, _vp(native.data_ptr()) if native is not None else None))

    def dslash_backfield(self, parity, out, inp, links, backfield):
        self._check(lib.lqcd_dslash_backfield(self._ctx, parity, _vp(out.data_ptr()), _vp(inp.data_ptr()),
                                              _vp(links.data_ptr()), _vp(backfield.data_ptr())))

    def dslash_slices(self, parity, out, inp, links, x3_lo, x3_hi):
        self._check(lib.lqcd_dslash_slices(self._ctx, parity, _vp(out.data_ptr()), _vp(inp.data_ptr()),
                                           _vp(links.data_ptr()), x3_lo, x3_hi))

    @property
    def halo_bytes(self):
        return int(lib.lqcd_halo_bytes(self._ctx))

    def halo_pack(self, buf, spinor_ptr, x3, sign=1.0):
        """spinor_ptr: a native half vector as a tensor or a raw device address."""
        ptr = spinor_ptr if isinstance(spinor_ptr, int) else spinor_ptr.data_ptr()
        self._check(lib.lqcd_halo_pack(self._ctx, _vp(buf.data_ptr()), _vp(ptr), x3, float(sign)))

    def halo_unpack(self, spinor_ptr, buf, x3):
        ptr = spinor_ptr if isinstance(spinor_ptr, int) else spinor_ptr.data_ptr()
        self._check(lib.lqcd_halo_unpack(self._ctx, _vp(ptr), _vp(buf.data_ptr()), x3))

    def halo_pack_faces(self, buf_top, buf_bottom, spinor_ptr, sign_top, sign_bottom):
        ptr = spinor_ptr if isinstance(spinor_ptr, int) else spinor_ptr.data_ptr()
        self._check(lib.lqcd_halo_pack_faces(self._ctx, _vp(buf_top.data_ptr()), _vp(buf_bottom.data_ptr()), _vp(ptr),
                                             float(sign_top), float(sign_bottom)))

    def halo_unpack_ghosts(self, spinor_ptr, buf_from_down, buf_from_up):
        ptr = spinor_ptr if isinstance(spinor_ptr, int) else spinor_ptr.data_ptr()
        self._check(lib.lqcd_halo_unpack_ghosts(self._ctx, _vp(ptr), _vp(buf_from_down.data_ptr()),
                                                _vp(buf_from_up.data_ptr())))

    def set_slab(self, x3_lo, x3_hi, solve_parity, halo_cb=None, allreduce_cb=None):
        """halo_cb / allreduce_cb: HALO_FN / ALLREDUCE_FN instances (kept alive here) or None."""
        self._slab_cbs = (halo_cb, allreduce_cb)
        self._check(lib.lqcd_set_slab(self._ctx, x3_lo, x3_hi, solve_parity,
                                      halo_cb if halo_cb is not None else HALO_FN(),
                                      allreduce_cb if allreduce_cb is not None else ALLREDUCE_FN(), None))

    # -- slab mode over the peer transport (lqcd_peer_*) ------------------------------------------------
    def peer_init(self, nranks, rank, x3_lo, x3_hi, solve_parity, sign_up, sign_down):
        """allocate this rank's block; returns its device address."""
        blk = _vp()
        self._check(lib.lqcd_peer_init(self._ctx, nranks, rank, x3_lo, x3_hi, solve_parity, float(sign_up),
                                       float(sign_down), C.byref(blk)))
        return int(blk.value)

    def peer_export(self):
        """64-byte CUDA IPC handle of this rank's block."""
        h = C.create_string_buffer(64)
        self._check(lib.lqcd_peer_export(self._ctx, h))
        return h.raw

    def peer_import(self, rank, handle):
        blk = _vp()
        self._check(lib.lqcd_peer_import(self._ctx, rank, C.create_string_buffer(bytes(handle), 64), C.byref(blk)))
        return int(blk.value)

    def peer_connect(self, blocks):
        arr = (_vp * len(blocks))(*[int(b) if b else None for b in blocks])
        self._check(lib.lqcd_peer_connect(self._ctx, arr))

    def peer_disconnect(self):
        self._check(lib.lqcd_peer_disconnect(self._ctx))

    def peer_selftest(self, nranks, rounds, sabotage=False):
        """protocol self-test under real concurrency (one cooperative kernel, CTA r = rank r); returns failures."""
        f = C.c_int(-1)
        self._check(lib.lqcd_peer_selftest(self._ctx, nranks, rounds, int(bool(sabotage)), C.byref(f)))
        return f.value

    def set_phase_hook(self, cb=None):
        """cb: a PHASE_FN instance (kept alive here) or None."""
        self._phase_cb = cb
        self._check(lib.lqcd_set_phase_hook(self._ctx, cb if cb is not None else PHASE_FN(), None))

    def mdagm(self, out_e, in_e, links, mass, sigma=0.0):
        self.ensure_workspace(1)
        self._check(lib.lqcd_mdagm(self._ctx, _vp(out_e.data_ptr()), _vp(in_e.data_ptr()), _vp(links.data_ptr()), mass, sigma))

    def mdagm_noalloc(self, out_e, in_e, links, mass, sigma=0.0):
        """mdagm without a workspace: the temporary is the library's fixed 8 MiB device array (lqcd.h).  No torch
        allocation happens here either; lattices whose half vector exceeds NOALLOC_SCRATCH_BYTES raise LqcdError."""
        self._check(lib.lqcd_mdagm_noalloc(self._ctx, _vp(out_e.data_ptr()), _vp(in_e.data_ptr()), _vp(links.data_ptr()),
                                           mass, sigma))

    def cg(self, x_e, b_e, links, mass, tol, max_iter, raise_on_max_iter=True):
        """blocking; returns dict(iters, rel_resid, converged)."""
        self.ensure_workspace(1)
        iters, res = C.c_int(0), C.c_double(0.0)
        rc = self._check(lib.lqcd_cg(self._ctx, _vp(x_e.data_ptr()), _vp(b_e.data_ptr()), _vp(links.data_ptr()),
                                     mass, tol, max_iter, C.byref(iters), C.byref(res)),
                         allow=() if raise_on_max_iter else (ERR_NOT_CONVERGED,))
        return dict(iters=iters.value, rel_resid=res.value, converged=(rc == OK))

    def cg_multishift(self, xs, b_e, links, mass, shifts, tol, max_iter, raise_on_max_iter=True):
        """blocking; xs: list of native even-site buffers (outputs)."""
        import numpy as np
        n = len(xs)
        self.ensure_workspace(n)
        sh = np.ascontiguousarray(shifts, dtype=np.float64)
        assert sh.size == n
        ptrs = (_vp * n)(*[x.data_ptr() for x in xs])
        iters = C.c_int(0)
        conv = (C.c_int * n)()
        res = np.zeros(n)
        rc = self._check(lib.lqcd_cg_multishift(self._ctx, n, sh.ctypes.data_as(_pd), _vp(b_e.data_ptr()), ptrs,
                                                _vp(links.data_ptr()), mass, tol, max_iter, C.byref(iters), conv,
                                                res.ctypes.data_as(_pd)),
                         allow=() if raise_on_max_iter else (ERR_NOT_CONVERGED,))
        return dict(iters=iters.value, conv_iter=np.array(list(conv)), rel_resid=res, converged=(rc == OK))

    def rational_apply(self, y_e, b_e, links, mass, shifts, c0, coeffs, tol, max_iter, raise_on_max_iter=True):
        """blocking; y = c0 b + sum_i coeffs[i] (A + shifts[i])^-1 b, accumulated inside the solve."""
        import numpy as np
        sh = np.ascontiguousarray(shifts, dtype=np.float64)
        co = np.ascontiguousarray(coeffs, dtype=np.float64)
        n = sh.size
        assert co.size == n
        self.ensure_workspace(n)
        iters = C.c_int(0)
        conv = (C.c_int * n)()
        rc = self._check(lib.lqcd_rational_apply(self._ctx, n, sh.ctypes.data_as(_pd), float(c0), co.ctypes.data_as(_pd),
                                                 _vp(b_e.data_ptr()), _vp(y_e.data_ptr()), _vp(links.data_ptr()),
                                                 mass, tol, max_iter, C.byref(iters), conv),
                         allow=() if raise_on_max_iter else (ERR_NOT_CONVERGED,))
        return dict(iters=iters.value, conv_iter=np.array(list(conv)), converged=(rc == OK))

    def fermion_force(self, xs, links, coeffs, force=None):
        """async; xs: the solutions x_i (native even-site buffers); returns the native (tamat) force buffer."""
        import numpy as np
        n = len(xs)
        co = np.ascontiguousarray(coeffs, dtype=np.float64)
        assert co.size == n
        self.ensure_workspace(n)
        if force is None:
            force = self._buf(int(lib.lqcd_tamat_bytes(self._ctx)))
        ptrs = (_vp * n)(*[x.data_ptr() for x in xs])
        self._check(lib.lqcd_fermion_force(self._ctx, n, co.ctypes.data_as(_pd), ptrs, _vp(links.data_ptr()),
                                           _vp(force.data_ptr())))
        return force

    def gauge_staples(self, links, c0=5.0 / 3.0, c1=-1.0 / 12.0, out=None):
        """async; tree-level Symanzik staples (3x3 per link); read back with unpack_force."""
        if out is None:
            out = self._buf(int(lib.lqcd_force_bytes(self._ctx)))
        if self.get_option("staples_variant") == 2:     # the two-pass algorithm keeps its 3-link staples in the workspace
            self.ensure_workspace(1, int(lib.lqcd_staples_workspace_bytes(self._ctx)))
        self._check(lib.lqcd_gauge_staples(self._ctx, _vp(links.data_ptr()), _vp(out.data_ptr()), float(c0), float(c1)))
        return out

    def unpack_tamat(self, native):
        """native 8-real (tamat) field, e.g. the fermion force -> numpy complex128 [V][4][3][3]."""
        import numpy as np
        canon = self.torch.empty(self.V * 4 * 9 * 2, dtype=self.torch.float64, device=self.device)
        self._check(lib.lqcd_unpack_tamat(self._ctx, _vp(canon.data_ptr()), _vp(native.data_ptr())))
        self.synchronize()
        return canon.cpu().numpy().view(np.complex128).reshape(self.V, 4, 3, 3)

    def unpack_force(self, native):
        """native 3x3-per-link field (gauge staples) -> numpy complex128 [V][4][3][3]."""
        import numpy as np
        canon = self.torch.empty(self.V * 4 * 9 * 2, dtype=self.torch.float64, device=self.device)
        self._check(lib.lqcd_unpack_force(self._ctx, _vp(canon.data_ptr()), _vp(native.data_ptr())))
        self.synchronize()
        return canon.cpu().numpy().view(np.complex128).reshape(self.V, 4, 3, 3)

    def solver_history(self):
        import numpy as np
        a, b, r = np.zeros(64), np.zeros(64), np.zeros(64)
        n = lib.lqcd_solver_history(self._ctx, 64, a.ctypes.data_as(_pd), b.ctypes.data_as(_pd), r.ctypes.data_as(_pd))
        n = max(0, min(n, 64))
        return dict(alpha=a[:n], beta=b[:n], rnorm=r[:n])

    # -- end-to-end on host buffers (blocking) --------------------------------------------------
    def dslash_host(self, parity, out_host, in_host, links_host):
        """numpy complex128 arrays (pinned or not); copies + pack + kernel + unpack inside the call."""
        self._check(lib.lqcd_dslash_host(self._ctx, parity, _vp(out_host.ctypes.data), _vp(in_host.ctypes.data),
                                         _vp(links_host.ctypes.data)))

    def dslash_host_vectors(self, parity, out_host, in_host, links):
        """as dslash_host, links resident on the device in native form (only the vectors are copied)."""
        self._check(lib.lqcd_dslash_host_vectors(self._ctx, parity, _vp(out_host.ctypes.data), _vp(in_host.ctypes.data),
                                                 _vp(links.data_ptr())))

    def cg_multishift_host(self, sol_host, rhs_host, links_host, mass, shifts, tol, max_iter, raise_on_max_iter=True):
        import numpy as np
        sh = np.ascontiguousarray(shifts, dtype=np.float64)
        n = sh.size
        iters = C.c_int(0)
        conv = (C.c_int * n)()
        res = np.zeros(n)
        rc = self._check(lib.lqcd_cg_multishift_host(self._ctx, n, sh.ctypes.data_as(_pd), _vp(rhs_host.ctypes.data),
                                                     _vp(sol_host.ctypes.data), _vp(links_host.ctypes.data), mass, tol,
                                                     max_iter, C.byref(iters), conv, res.ctypes.data_as(_pd)),
                         allow=() if raise_on_max_iter else (ERR_NOT_CONVERGED,))
        return dict(iters=iters.value, conv_iter=np.array(list(conv)), rel_resid=res, converged=(rc == OK))

    def dslash_host_vectors_batch(self, parities, outs_host, ins_host, links):
        """n applications on host vectors in one pipelined call (uploads, compute and downloads overlap)."""
        n = len(parities)
        assert len(outs_host) == n and len(ins_host) == n
        par = (C.c_int * n)(*[int(p) for p in parities])
        outs = (_vp * n)(*[o.ctypes.data for o in outs_host])
        ins = (_vp * n)(*[i.ctypes.data for i in ins_host])
        self._check(lib.lqcd_dslash_host_vectors_batch(self._ctx, n, par, outs, ins, _vp(links.data_ptr())))

    def cg_multishift_host_vectors(self, sol_host, rhs_host, links, mass, shifts, tol, max_iter, raise_on_max_iter=True):
        """as cg_multishift_host with the links resident on the device in native form."""
        import numpy as np
        sh = np.ascontiguousarray(shifts, dtype=np.float64)
        n = sh.size
        self.ensure_workspace(n)
        iters = C.c_int(0)
        conv = (C.c_int * n)()
        res = np.zeros(n)
        rc = self._check(lib.lqcd_cg_multishift_host_vectors(self._ctx, n, sh.ctypes.data_as(_pd), _vp(rhs_host.ctypes.data),
                                                             _vp(sol_host.ctypes.data), _vp(links.data_ptr()), mass, tol,
                                                             max_iter, C.byref(iters), conv, res.ctypes.data_as(_pd)),
                         allow=() if raise_on_max_iter else (ERR_NOT_CONVERGED,))
        return dict(iters=iters.value, conv_iter=np.array(list(conv)), rel_resid=res, converged=(rc == OK))

    def measure_hbm_read(self, buf):
        """attainable read bandwidth in GB/s over a device buffer larger than L2 (measurement helper; blocking)."""
        v = C.c_double(0.0)
        self._check(lib.lqcd_measure_hbm_read(self._ctx, _vp(buf.data_ptr()), buf.numel() * buf.element_size(), C.byref(v)))
        return v.value

    def measure_fp64_peak(self):
        """attainable FP64 FMA rate in TFLOP/s (measurement helper; blocking)."""
        v = C.c_double(0.0)
        self._check(lib.lqcd_measure_fp64_peak(self._ctx, C.byref(v)))
        return v.value
