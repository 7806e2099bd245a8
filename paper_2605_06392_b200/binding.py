"""ctypes binding with the same names as include/bta.h (and include/bta_diag.h).  Marshalling only."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))


def lib_path() -> str:
    return os.path.join(_HERE, "libbta_b200.so")


class BtaError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"bta error {code}: {msg}")
        self.code = code


class _Desc(C.Structure):
    _fields_ = [("nt", C.c_int32), ("g", C.c_int32), ("k", C.c_int32), ("a", C.c_int32),
                ("h", C.c_double), ("fixed_prec", C.c_double)]


class _Obs(C.Structure):
    _fields_ = [("m", C.c_int64), ("var", C.c_void_p), ("node", C.c_void_p), ("time", C.c_void_p),
                ("cov", C.c_void_p), ("y", C.c_void_p)]


class _Blocks(C.Structure):
    _fields_ = [("D", C.c_void_p), ("B", C.c_void_p), ("C", C.c_void_p), ("T", C.c_void_p), ("rhs", C.c_void_p)]


_lib = None


def lib():
    """Load libbta_b200.so (built in-tree by build.py); fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -m paper_2605_06392_b200.build` "
                          "(or __graft_entry__.build()); there is no fallback path")
    L = C.CDLL(path)
    vp, dp, i32, i64 = C.c_void_p, C.POINTER(C.c_double), C.c_int, C.c_int64
    L.bta_create.argtypes = [C.POINTER(vp), C.POINTER(_Desc), C.POINTER(_Obs), i32]
    L.bta_destroy.argtypes = [vp]
    L.bta_workspace_bytes.argtypes = [vp]
    L.bta_workspace_bytes.restype = C.c_size_t
    L.bta_workspace_bytes_op.argtypes = [vp]
    L.bta_workspace_bytes_op.restype = C.c_size_t
    L.bta_assemble.argtypes = [vp, dp, i32, _Blocks, vp]
    L.bta_factor_logdet.argtypes = [vp, _Blocks, i32, dp, vp, vp, vp]
    L.bta_solve.argtypes = [vp, _Blocks, i32, vp, i32, vp, vp]
    L.bta_selinv.argtypes = [vp, _Blocks, i32, vp, vp]
    L.inla_value_and_grad.argtypes = [vp, dp, dp, dp, dp, vp, vp]
    L.inla_value.argtypes = [vp, dp, dp, vp, vp]
    L.inla_fd_grad.argtypes = [vp, dp, C.c_double, dp, dp, vp, vp]
    L.inla_hessian.argtypes = [vp, dp, C.c_double, dp, dp, dp, vp, vp]
    L.inla_optimize.argtypes = [vp, dp, i32, C.c_double, dp, dp, dp, C.POINTER(C.c_int), C.POINTER(C.c_int), vp, vp]
    L.bta_last_intermediates.argtypes = [vp, dp, dp, dp, dp, dp, dp]
    L.bta_num_hyper.argtypes = [vp]
    L.bta_num_hyper.restype = C.c_int32
    L.bta_latent_size.argtypes = [vp]
    L.bta_latent_size.restype = i64
    L.bta_last_pivot.argtypes = [vp]
    L.bta_last_pivot.restype = i64
    L.bta_kernel_launches.argtypes = [vp]
    L.bta_kernel_launches.restype = i64
    L.bta_last_error.restype = C.c_char_p
    L.bta_set_store_mode.argtypes = [vp, i32]
    L.bta_host_bytes.argtypes = [vp]
    L.bta_host_bytes.restype = C.c_size_t
    L.bta_set_host_buffer.argtypes = [vp, vp, C.c_size_t]
    L.bta_get_store_mode.argtypes = [vp]
    L.bta_fp64_peak.argtypes = [i32, i32, dp, dp, vp]
    L.bta_gemm.argtypes = [i32, i32, i32, i32, C.c_double, vp, i32, vp, i32, C.c_double, vp, i32, i32, i32, i32, vp]
    L.bta_debug_cta_trace.argtypes = [vp, C.c_uint]
    L.bta_debug_cta_trace_count.argtypes = [C.POINTER(C.c_uint)]
    L.bta_diag_gemm_flop.argtypes = [i32, i32, i32, i32, i32, i32]
    L.bta_diag_gemm_flop.restype = C.c_double
    L.bta_diag_ktime_begin.argtypes = []
    L.bta_diag_ktime_end.argtypes = [dp, dp, dp, C.POINTER(C.c_int64)]
    L.bta_partition_plan.argtypes = [vp, i32, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    L.bta_part_slab_doubles.argtypes = [vp]
    L.bta_part_slab_doubles.restype = C.c_size_t
    L.bta_part_partial_doubles.argtypes = [vp]
    L.bta_part_partial_doubles.restype = C.c_size_t
    L.inla_part_phase1.argtypes = [vp, dp, i32, i32, vp, vp, vp]
    L.inla_part_phase2.argtypes = [vp, i32, i32, vp, vp, vp, vp]
    L.inla_part_finish.argtypes = [vp, vp, dp, dp, vp]
    rtb = [i32, i32, i32, vp, i32, vp, i32, i32, C.c_double, C.c_double, vp, i32, vp, i32]
    L.bta_rows_times_block_noalloc.argtypes = rtb + [vp]
    L.bta_rows_times_block.argtypes = rtb + [vp, vp]
    L.bta_rows_times_block_t.argtypes = rtb + [vp]
    L.bta_diag_potrf_inv.argtypes = [vp, vp, i32, i32, vp, vp, vp, vp]
    L.bta_set_option.argtypes = [vp, i32, i32]
    L.bta_get_option.argtypes = [vp, i32]
    _lib = L
    return L


def _check(rc):
    if rc != 0:
        raise BtaError(rc, lib().bta_last_error().decode())


def _dptr(arr):
    return arr.ctypes.data_as(C.POINTER(C.c_double))


def _stream():
    import torch
    return torch.cuda.current_stream().cuda_stream


@dataclass
class Blocks:
    """Device tensors of one BTA matrix (layouts of include/bta.h)."""
    D: object
    B: object
    C: object
    T: object
    rhs: object = None

    def c(self):
        p = lambda t: t.data_ptr() if t is not None and t.numel() > 0 else None
        return _Blocks(p(self.D), p(self.B), p(self.C), p(self.T), p(self.rhs))

    def clone(self):
        cl = lambda t: t.clone() if t is not None else None
        return Blocks(cl(self.D), cl(self.B), cl(self.C), cl(self.T), cl(self.rhs))


BTA_PRIOR, BTA_COND = 0, 1
BTA_STORE_FACTOR, BTA_STORE_CARRY, BTA_STORE_HOST = 0, 1, 2
OPT_TWIST, OPT_LANES, OPT_SPLIT, OPT_GRAPH, OPT_SERIAL, OPT_PIPELINE, OPT_TILE_THRESH, OPT_TILE_WAVES, OPT_PARTITIONS, OPT_PDL, OPT_ROWS = range(11)
STAGES = ("assemble", "fwd_Qc", "bwd_Qc", "fwd_Qp", "bwd_Qp", "scalars", "total")


class BtaModel:
    """bta_create / bta_destroy plus the calls of include/bta.h on torch-owned device memory."""

    def __init__(self, nt, g, k, a, h, fixed_prec, var, node, time, cov, y, device=0):
        import torch
        self._h = C.c_void_p()
        self.nt, self.g, self.k, self.a = int(nt), int(g), int(k), int(a)
        self.ns = self.g * self.g
        self.b = self.k * self.ns
        self.device = torch.device("cuda", device)
        var = np.ascontiguousarray(var, dtype=np.int32)
        node = np.ascontiguousarray(node, dtype=np.int32)
        time = np.ascontiguousarray(time, dtype=np.int32)
        cov = np.ascontiguousarray(cov, dtype=np.float64)
        y = np.ascontiguousarray(y, dtype=np.float64)
        desc = _Desc(self.nt, self.g, self.k, self.a, float(h), float(fixed_prec))
        obs = _Obs(int(y.shape[0]), var.ctypes.data, node.ctypes.data, time.ctypes.data, cov.ctypes.data, y.ctypes.data)
        _check(lib().bta_create(C.byref(self._h), C.byref(desc), C.byref(obs), device))
        self.d = lib().bta_num_hyper(self._h)
        self.N = lib().bta_latent_size(self._h)
        self._ws = None
        self._ws_op = None
        self._host = None

    @classmethod
    def from_workload(cls, model, obs, device=0):
        return cls(model.nt, model.g, model.k, model.a, model.h, model.fixed_prec, obs.var, obs.node, obs.time,
                   obs.cov, obs.y, device=device)

    def close(self):
        if self._h:
            lib().bta_destroy(self._h)
            self._h = C.c_void_p()
            self._ws = self._ws_op = self._host = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- memory (torch owns it) ----
    def workspace_bytes(self):
        return lib().bta_workspace_bytes(self._h)

    def workspace_bytes_op(self):
        return lib().bta_workspace_bytes_op(self._h)

    def _workspace(self, op=False):
        import torch
        if op:
            if self._ws_op is None:
                self._ws_op = torch.empty(self.workspace_bytes_op(), dtype=torch.uint8, device=self.device)
            return self._ws_op
        if self._ws is None:
            self._ws = torch.empty(self.workspace_bytes(), dtype=torch.uint8, device=self.device)
        return self._ws

    def alloc_blocks(self, rhs=True):
        import torch
        kw = dict(dtype=torch.float64, device=self.device)
        return Blocks(torch.empty(self.nt, self.b, self.b, **kw), torch.empty(max(self.nt - 1, 0), self.b, self.b, **kw),
                      torch.empty(self.nt, self.a, self.b, **kw), torch.empty(self.a, self.a, **kw),
                      torch.empty(self.N, **kw) if rhs else None)

    # ---- the calls of include/bta.h ----
    def bta_assemble(self, theta, which, out: Blocks):
        th = np.ascontiguousarray(theta, dtype=np.float64)
        assert th.shape == (self.d,)
        _check(lib().bta_assemble(self._h, _dptr(th), which, out.c(), _stream()))
        return out

    def bta_factor_logdet(self, blocks: Blocks, which, diagL=None):
        ld = C.c_double()
        _check(lib().bta_factor_logdet(self._h, blocks.c(), which, C.byref(ld),
                                       diagL.data_ptr() if diagL is not None else None,
                                       self._workspace(op=True).data_ptr(), _stream()))
        return ld.value

    def bta_solve(self, factor: Blocks, which, rhs):
        """rhs: device tensor [nrhs, N], solved in place."""
        assert rhs.is_contiguous() and rhs.shape[-1] == self.N
        nrhs = 1 if rhs.dim() == 1 else rhs.shape[0]
        _check(lib().bta_solve(self._h, factor.c(), which, rhs.data_ptr(), nrhs, self._workspace(op=True).data_ptr(),
                               _stream()))
        return rhs

    def bta_selinv(self, factor: Blocks, which):
        _check(lib().bta_selinv(self._h, factor.c(), which, self._workspace(op=True).data_ptr(), _stream()))
        return factor

    def inla_value_and_grad(self, theta, stages=False):
        th = np.ascontiguousarray(theta, dtype=np.float64)
        assert th.shape == (self.d,)
        f = C.c_double()
        grad = np.zeros(self.d)
        st = np.zeros(len(STAGES))
        _check(lib().inla_value_and_grad(self._h, _dptr(th), C.byref(f), _dptr(grad), _dptr(st) if stages else None,
                                         self._workspace().data_ptr(), _stream()))
        if stages:
            return f.value, grad, dict(zip(STAGES, st.tolist()))
        return f.value, grad

    def inla_value(self, theta):
        th = np.ascontiguousarray(theta, dtype=np.float64)
        f = C.c_double()
        _check(lib().inla_value(self._h, _dptr(th), C.byref(f), self._workspace().data_ptr(), _stream()))
        return f.value

    def inla_fd_grad(self, theta, h=1e-3):
        """Central finite differences of inla_value (Eq. 2): 2d+1 evaluations."""
        th = np.ascontiguousarray(theta, dtype=np.float64)
        f = C.c_double()
        g = np.zeros(self.d)
        _check(lib().inla_fd_grad(self._h, _dptr(th), float(h), C.byref(f), _dptr(g), self._workspace().data_ptr(),
                                  _stream()))
        return f.value, g

    def inla_hessian(self, theta, h=5e-3):
        """Central differences of the exact gradient (Eq. 13): 2d+1 gradient calls."""
        th = np.ascontiguousarray(theta, dtype=np.float64)
        f = C.c_double()
        g = np.zeros(self.d)
        H = np.zeros((self.d, self.d))
        _check(lib().inla_hessian(self._h, _dptr(th), float(h), C.byref(f), _dptr(g), _dptr(H),
                                  self._workspace().data_ptr(), _stream()))
        return f.value, g, H

    def inla_optimize(self, theta0, max_iter=100, gtol=1e-6):
        """L-BFGS mode search on f (maximisation); returns (theta*, f*, grad*, iterations, gradient evaluations)."""
        th0 = np.ascontiguousarray(theta0, dtype=np.float64)
        th = np.zeros(self.d)
        g = np.zeros(self.d)
        f = C.c_double()
        it, ev = C.c_int(), C.c_int()
        _check(lib().inla_optimize(self._h, _dptr(th0), int(max_iter), float(gtol), _dptr(th), C.byref(f), _dptr(g),
                                   C.byref(it), C.byref(ev), self._workspace().data_ptr(), _stream()))
        return th, f.value, g, it.value, ev.value

    def last_intermediates(self, want_x=True):
        ld = np.zeros(2)
        x = np.zeros(self.N) if want_x else None
        parts = np.zeros(3 * self.d)
        rss = np.zeros(self.k)
        quad = C.c_double()
        ZT = np.zeros((self.a, self.a))
        _check(lib().bta_last_intermediates(self._h, _dptr(ld), _dptr(x) if want_x else None, _dptr(parts), _dptr(rss),
                                            C.byref(quad), _dptr(ZT)))
        return dict(ZT=ZT, ld_p=ld[0], ld_c=ld[1], x=x, phaseA=parts[: self.d], phaseB=parts[self.d: 2 * self.d],
                    phaseC=parts[2 * self.d:], rss=rss, quad_p=quad.value)

    def bta_set_store_mode(self, mode):
        """BTA_STORE_FACTOR (0), BTA_STORE_CARRY (1) or BTA_STORE_HOST (2); the gradient workspace is re-sized on next
        use.  For BTA_STORE_HOST a pinned torch tensor of bta_host_bytes() is allocated and registered."""
        import torch
        _check(lib().bta_set_store_mode(self._h, int(mode)))
        self._ws = None
        if int(mode) == BTA_STORE_HOST:
            need = lib().bta_host_bytes(self._h)
            if need and (self._host is None or self._host.numel() < need):
                self._host = torch.empty(need, dtype=torch.uint8, pin_memory=True)
            if need:
                _check(lib().bta_set_host_buffer(self._h, self._host.data_ptr(), need))
        else:
            _check(lib().bta_set_host_buffer(self._h, None, 0))
            self._host = None

    def bta_host_bytes(self):
        return lib().bta_host_bytes(self._h)

    def bta_get_store_mode(self):
        return lib().bta_get_store_mode(self._h)

    def bta_set_option(self, option, value):
        """include/bta_diag.h: OPT_TWIST / OPT_LANES / OPT_SPLIT / OPT_GRAPH / OPT_SERIAL / OPT_PIPELINE."""
        _check(lib().bta_set_option(self._h, int(option), int(value)))

    def bta_get_option(self, option):
        return lib().bta_get_option(self._h, int(option))

    def bta_set_partitions(self, P):
        """P >= 2: time-domain partitioning with P partitions inside the GPU (0: two-way elimination).  Re-sizes the
        workspace."""
        self.bta_set_option(OPT_PARTITIONS, P)
        self._ws = None

    # ---- the multi-rank form of the partitioning (include/bta.h: inla_part_*); buffers are torch tensors
    def inla_part_phase1(self, theta, rank, nranks):
        """-> this rank's slab (device tensor, float64) for the all-gather."""
        import torch
        th = np.ascontiguousarray(theta, dtype=np.float64)
        slab = torch.zeros(lib().bta_part_slab_doubles(self._h), dtype=torch.float64, device=self.device)
        _check(lib().inla_part_phase1(self._h, _dptr(th), int(rank), int(nranks), slab.data_ptr(),
                                      self._workspace().data_ptr(), _stream()))
        return slab

    def inla_part_phase2(self, rank, nranks, gathered):
        """gathered: device tensor of nranks slabs in rank order -> this rank's partial sums (device tensor)."""
        import torch
        assert gathered.is_contiguous() and gathered.numel() == nranks * lib().bta_part_slab_doubles(self._h)
        partials = torch.empty(lib().bta_part_partial_doubles(self._h), dtype=torch.float64, device=self.device)
        _check(lib().inla_part_phase2(self._h, int(rank), int(nranks), gathered.data_ptr(), partials.data_ptr(),
                                      self._workspace().data_ptr(), _stream()))
        return partials

    def inla_part_finish(self, partials):
        """partials: the all-reduced partial sums -> (f, grad)."""
        f = C.c_double()
        grad = np.zeros(self.d)
        _check(lib().inla_part_finish(self._h, partials.data_ptr(), C.byref(f), _dptr(grad), _stream()))
        return f.value, grad

    def bta_partition_plan(self, P):
        """-> [(first, last)] time blocks of the partitions a request for P partitions yields."""
        first = (C.c_int32 * 8)()
        last = (C.c_int32 * 8)()
        n = lib().bta_partition_plan(self._h, int(P), first, last)
        return [(first[i], last[i]) for i in range(n)]

    def kernel_launches(self):
        return lib().bta_kernel_launches(self._h)

    def last_pivot(self):
        return lib().bta_last_pivot(self._h)

    def diag_potrf_inv(self, A, diagL=None):
        """include/bta_diag.h: A (device, n x n, lower, SPD) -> chol(A)^-1 in place, as the forward sweeps do it."""
        import torch
        n = A.shape[0]
        T1, T2 = torch.empty_like(A), torch.empty_like(A)
        _check(lib().bta_diag_potrf_inv(self._h, A.data_ptr(), A.stride(0), n, T1.data_ptr(), T2.data_ptr(),
                                        diagL.data_ptr() if diagL is not None else None, _stream()))
        return A


def fp64_peak(kind=0, iters=100000):
    """(TFLOP/s, ms) of the register-resident DMMA (kind 0) or DFMA (kind 1) issue loop."""
    tf, ms = C.c_double(), C.c_double()
    _check(lib().bta_fp64_peak(kind, iters, C.byref(tf), C.byref(ms), _stream()))
    return tf.value, ms.value


def gemm(mode, A, B, Cm, alpha=1.0, beta=0.0, klo=0, khi=0, out=0):
    """C = alpha op(A) op(B) + beta C through the library's DMMA GEMM (device tensors, row-major)."""
    if mode == 0:
        M, K = A.shape
        N = B.shape[1]
    elif mode == 1:
        M, K = A.shape
        N = B.shape[0]
    else:
        K, M = A.shape
        N = B.shape[1]
    _check(lib().bta_gemm(mode, M, N, K, alpha, A.data_ptr(), A.stride(0), B.data_ptr(), B.stride(0), beta,
                          Cm.data_ptr(), Cm.stride(0), klo, khi, out, _stream()))
    return Cm


KCLASSES = ("gemm_128", "gemm_64", "gemm_32", "leaf", "skinny", "contract", "assemble", "other")


def ktime_begin():
    """include/bta_diag.h: arm the per-kernel-class timing (every launch bracketed by CUDA events)."""
    _check(lib().bta_diag_ktime_begin())


def ktime_end():
    """-> {class: dict(ms, flop, bytes, launches)} of the launches since ktime_begin (synchronises the device)."""
    n = len(KCLASSES)
    ms, fl, by = np.zeros(n), np.zeros(n), np.zeros(n)
    cnt = np.zeros(n, dtype=np.int64)
    _check(lib().bta_diag_ktime_end(_dptr(ms), _dptr(fl), _dptr(by), cnt.ctypes.data_as(C.POINTER(C.c_int64))))
    return {k: dict(ms=float(ms[i]), flop=float(fl[i]), bytes=float(by[i]), launches=int(cnt[i]))
            for i, k in enumerate(KCLASSES)}


def gemm_alg_flop(M, N, K, klo=0, khi=0, out=0):
    return lib().bta_diag_gemm_flop(M, N, K, klo, khi, out)


NOALLOC_MAX_PART = 32 * 9 * 4096


def rows_times_block_noalloc(R, M, out, alpha=1.0, beta=0.0, inp=None, tri=0):
    """out = alpha R M + beta inp with the kernel's scratch in the library's static device array (include/bta.h)."""
    P, K = R.shape
    J = M.shape[1]
    _check(lib().bta_rows_times_block_noalloc(P, K, J, R.data_ptr(), R.stride(0), M.data_ptr(), M.stride(0), int(tri),
                                              alpha, beta, inp.data_ptr() if inp is not None else None,
                                              inp.stride(0) if inp is not None else 0, out.data_ptr(), out.stride(0),
                                              _stream()))
    return out


def rows_times_block(R, M, out, part, alpha=1.0, beta=0.0, inp=None, tri=0):
    """The same product through the sweeps' launcher with caller-provided scratch (include/bta_diag.h)."""
    P, K = R.shape
    J = M.shape[1]
    _check(lib().bta_rows_times_block(P, K, J, R.data_ptr(), R.stride(0), M.data_ptr(), M.stride(0), int(tri), alpha,
                                      beta, inp.data_ptr() if inp is not None else None,
                                      inp.stride(0) if inp is not None else 0, out.data_ptr(), out.stride(0),
                                      part.data_ptr(), _stream()))
    return out


def rows_times_block_t(R, M, out, alpha=1.0, beta=0.0, inp=None, tri=0):
    """out = alpha R M^T + beta inp (k <= j only when tri): the forward sweeps' skinny product (include/bta_diag.h)."""
    P, K = R.shape
    J = M.shape[0]
    _check(lib().bta_rows_times_block_t(P, J, K, R.data_ptr(), R.stride(0), M.data_ptr(), M.stride(0), int(tri), alpha,
                                        beta, inp.data_ptr() if inp is not None else None,
                                        inp.stride(0) if inp is not None else 0, out.data_ptr(), out.stride(0), _stream()))
    return out


def cta_trace_start(buf):
    """Diagnostic: arm the per-CTA GEMM timeline; `buf` is a CUDA int64 tensor of shape [cap, 4] (None: off)."""
    if buf is None:
        _check(lib().bta_debug_cta_trace(None, 0))
    else:
        _check(lib().bta_debug_cta_trace(buf.data_ptr(), buf.shape[0]))


def cta_trace_count():
    n = C.c_uint(0)
    _check(lib().bta_debug_cta_trace_count(C.byref(n)))
    return n.value
