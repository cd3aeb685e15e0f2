"""Thin ctypes binding of libsubmatrix_b200.so -- same names as include/submatrix.h.

Argument marshalling only: PyTorch provides device memory and the CUDA stream, every step of the
path (index build, gather, Newton-Schulz, scatter, traces, bisection) runs inside the library.
There is NO CPU fallback: importing this module without the built library raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsubmatrix_b200.so")

SM_OK = 0
SM_ERR_INVALID_ARG = -1
SM_ERR_STRUCTURE = -2
SM_ERR_ALLOC = -3
SM_ERR_CUDA = -4
SM_ERR_WORKSPACE_TOO_SMALL = -5
SM_WARN_SIGN_NOT_CONVERGED = 1
SM_WARN_MU_NOT_CONVERGED = 2

EXPORTS = [
    "sm_plan_create", "sm_plan_query", "sm_plan_export_index", "sm_sign_execute", "sm_sign_execute_host",
    "sm_density_matrix", "sm_density_matrix_host", "sm_trace_dk", "sm_gather", "sm_sign_iterate",
    "sm_scatter", "sm_set_timing", "sm_launch_count", "sm_plan_destroy", "sm_strerror",
    "sm_last_cuda_error", "sm_measure_peaks", "sm_eig_decompose", "sm_eig_export", "sm_eig_nelec", "sm_eig_density",
    "sm_partition_groups", "sm_plan_set_allreduce", "sm_trace_dk_static",
]


class sm_options_t(C.Structure):
    _fields_ = [("max_iter", C.c_int32), ("scaling", C.c_int32), ("precision", C.c_int32),
                ("check_every", C.c_int32), ("max_mu_steps", C.c_int32), ("bisect_iter", C.c_int32),
                ("mu_tol", C.c_double), ("early_out", C.c_int32), ("order", C.c_int32),
                ("overshoot", C.c_double), ("predict", C.c_int32), ("mu_guess", C.c_int32), ("rescale", C.c_int32), ("mu_start", C.c_int32),
                ("method", C.c_int32), ("reserved1", C.c_int32), ("kT", C.c_double),
                ("shard_rank", C.c_int32), ("shard_world", C.c_int32)]


class sm_plan_info_t(C.Structure):
    _fields_ = [("nb", C.c_int32), ("ngroups", C.c_int32), ("nnzb", C.c_int64), ("nnz", C.c_int64),
                ("n_basis", C.c_int64), ("sum_sub_blocks", C.c_int64), ("dim_min", C.c_int32),
                ("dim_max", C.c_int32), ("dim_mean", C.c_double), ("sum_n2", C.c_int64), ("sum_n3", C.c_int64),
                ("sum_ld2", C.c_int64), ("n_tiles", C.c_int64), ("n_buckets", C.c_int32),
                ("reserved0", C.c_int32), ("workspace_bytes", C.c_size_t), ("sum_n3_columns", C.c_int64),
                ("est_speedup", C.c_double), ("index_alg_bytes", C.c_int64), ("ms_index_kernels", C.c_float),
                ("ms_plan_create", C.c_float), ("shard_group_begin", C.c_int32), ("shard_group_end", C.c_int32),
                ("shard_val_begin", C.c_int64), ("shard_val_end", C.c_int64), ("ngroups_total", C.c_int32),
                ("reserved2", C.c_int32)]


ALLREDUCE_FN = C.CFUNCTYPE(None, C.c_void_p, C.POINTER(C.c_double), C.c_int32)


class sm_peaks_t(C.Structure):
    _fields_ = [("dmma_tflops", C.c_double), ("hbm_copy_gbs", C.c_double), ("ms_dmma", C.c_double),
                ("ms_copy", C.c_double), ("num_sms", C.c_int32), ("reserved", C.c_int32)]


class sm_stats_t(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("iter_min", C.c_int32), ("iter_max", C.c_int32),
                ("not_converged", C.c_int32), ("max_residual", C.c_double), ("n_elec", C.c_double),
                ("mu", C.c_double), ("mu_steps", C.c_int32), ("gemm_launches", C.c_int32),
                ("sum_iter_n3", C.c_int64), ("ms_gather", C.c_float), ("ms_sign", C.c_float),
                ("ms_scatter", C.c_float), ("ms_total", C.c_float), ("mu_trace", C.c_double * 64),
                ("ne_trace", C.c_double * 64), ("ne_err_trace", C.c_double * 64), ("iter_trace", C.c_int32 * 64),
                ("tot_sum_iter_n3", C.c_int64), ("tot_sym_flop", C.c_int64),
                ("tot_gemm_launches", C.c_int32), ("tot_evaluations", C.c_int32),
                ("tot_ms_gather", C.c_float), ("tot_ms_sign", C.c_float),
                ("spec_lo", C.c_double), ("spec_hi", C.c_double), ("bracket_lo", C.c_double),
                ("bracket_hi", C.c_double), ("mu_guess", C.c_double),
                ("exits_predicted", C.c_int32), ("exits_two_step", C.c_int32),
                ("ms_gemm", C.c_float), ("tot_ms_gemm", C.c_float)]

    def as_dict(self):
        d = {k: getattr(self, k) for k, _ in self._fields_ if k not in ("mu_trace", "ne_trace", "ne_err_trace", "iter_trace")}
        n = max(int(self.mu_steps), 0)
        d["mu_trace"] = list(self.mu_trace[:n])
        d["ne_trace"] = list(self.ne_trace[:n])
        d["ne_err_trace"] = list(self.ne_err_trace[:n])
        d["iter_trace"] = list(self.iter_trace[:n])
        return d


def default_options(**kw) -> sm_options_t:
    o = sm_options_t(max_iter=100, scaling=1, precision=0, check_every=16, max_mu_steps=64, bisect_iter=0,
                     mu_tol=1e-6, early_out=1, overshoot=1.45, order=2, predict=2, mu_guess=1, rescale=1, mu_start=1,
                     method=0, reserved1=0, kT=0.0, shard_rank=0, shard_world=1)
    for k, v in kw.items():
        setattr(o, k, v)
    return o


_lib = None


def lib() -> C.CDLL:
    """Load the CUDA library; fails loudly if it was not built (no fallback exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2004_10811_b200.build` "
                               "(there is no CPU fallback for the submatrix hot path)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        L.sm_plan_create.argtypes = [C.POINTER(vp), i32, vp, vp, vp, i32, vp, vp, C.POINTER(sm_options_t), vp]
        L.sm_plan_query.argtypes = [vp, C.POINTER(sm_plan_info_t)]
        L.sm_plan_export_index.argtypes = [vp, vp, vp, vp, vp, vp]
        L.sm_sign_execute.argtypes = [vp, vp, dbl, dbl, vp, vp, C.c_size_t, C.POINTER(sm_stats_t), vp]
        L.sm_sign_execute_host.argtypes = L.sm_sign_execute.argtypes
        L.sm_density_matrix.argtypes = [vp, vp, dbl, dbl, dbl, C.POINTER(dbl), vp, vp, C.c_size_t,
                                        C.POINTER(sm_stats_t), vp]
        L.sm_density_matrix_host.argtypes = L.sm_density_matrix.argtypes
        L.sm_trace_dk.argtypes = [vp, vp, vp, C.POINTER(dbl), C.POINTER(dbl), vp]
        L.sm_trace_dk_static.argtypes = [C.c_int64, vp, vp, vp, vp]
        L.sm_gather.argtypes = [vp, vp, dbl, vp, C.c_size_t, vp]
        L.sm_sign_iterate.argtypes = [vp, dbl, vp, C.c_size_t, C.POINTER(sm_stats_t), vp]
        L.sm_scatter.argtypes = [vp, i32, vp, vp, C.c_size_t, vp]
        L.sm_set_timing.argtypes = [vp, i32]
        L.sm_launch_count.argtypes = [vp]
        L.sm_launch_count.restype = i64
        L.sm_plan_destroy.argtypes = [vp]
        L.sm_plan_destroy.restype = None
        L.sm_strerror.argtypes = [i32]
        L.sm_strerror.restype = C.c_char_p
        L.sm_last_cuda_error.restype = C.c_char_p
        L.sm_measure_peaks.argtypes = [C.POINTER(sm_peaks_t), vp]
        L.sm_eig_decompose.argtypes = [vp, vp, vp, C.c_size_t, C.POINTER(sm_stats_t), vp]
        L.sm_eig_export.argtypes = [vp, vp, vp, vp]
        L.sm_eig_nelec.argtypes = [vp, dbl, dbl, C.POINTER(dbl), vp]
        L.sm_eig_density.argtypes = [vp, dbl, dbl, vp, vp, C.c_size_t, vp]
        L.sm_partition_groups.argtypes = [i32, vp, i32, vp]
        L.sm_plan_set_allreduce.argtypes = [vp, ALLREDUCE_FN, vp]
        for f in ("sm_plan_create", "sm_plan_query", "sm_plan_export_index", "sm_sign_execute",
                  "sm_sign_execute_host", "sm_density_matrix", "sm_density_matrix_host", "sm_trace_dk",
                  "sm_gather", "sm_sign_iterate", "sm_scatter", "sm_set_timing", "sm_measure_peaks", "sm_eig_decompose", "sm_eig_export",
                  "sm_eig_nelec", "sm_eig_density", "sm_partition_groups", "sm_plan_set_allreduce"):
            getattr(L, f).restype = i32
        _lib = L
    return _lib


class SubmatrixError(RuntimeError):
    def __init__(self, status: int):
        L = lib()
        msg = L.sm_strerror(status).decode()
        if status == SM_ERR_CUDA:
            msg += " (" + L.sm_last_cuda_error().decode() + ")"
        super().__init__(f"sm status {status}: {msg}")
        self.status = status


def _check(status: int) -> int:
    if status < 0:
        raise SubmatrixError(status)
    return status


def _np_ptr(a):
    return a.ctypes.data if a is not None else None


def _dev_ptr(t):
    return None if t is None else t.data_ptr()


def _stream_ptr(stream=None):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return s.cuda_stream


# ------------------------------------------------------------------ functions (names of the C-ABI)
def sm_plan_create(nb, blk_size, colptr, rowidx, ngroups, grp_ptr, grp_cols, opt=None, stream=None):
    """-> opaque plan handle (int).  Host numpy arrays in, see include/submatrix.h."""
    blk_size = np.ascontiguousarray(blk_size, dtype=np.int32)
    colptr = np.ascontiguousarray(colptr, dtype=np.int64)
    rowidx = np.ascontiguousarray(rowidx, dtype=np.int32)
    grp_ptr = np.ascontiguousarray(grp_ptr, dtype=np.int32)
    grp_cols = np.ascontiguousarray(grp_cols, dtype=np.int32)
    h = C.c_void_p()
    _check(lib().sm_plan_create(C.byref(h), nb, _np_ptr(blk_size), _np_ptr(colptr), _np_ptr(rowidx), ngroups,
                                _np_ptr(grp_ptr), _np_ptr(grp_cols), C.byref(opt) if opt is not None else None,
                                _stream_ptr(stream)))
    return h


def sm_plan_query(plan) -> sm_plan_info_t:
    info = sm_plan_info_t()
    _check(lib().sm_plan_query(plan, C.byref(info)))
    return info


def sm_plan_export_index(plan):
    info = sm_plan_query(plan)
    sub_ptr = np.zeros(info.ngroups + 1, dtype=np.int64)
    sub_blocks = np.zeros(info.sum_sub_blocks, dtype=np.int32)
    sub_off = np.zeros(info.sum_sub_blocks, dtype=np.int32)
    sub_dim = np.zeros(info.ngroups, dtype=np.int32)
    gen_pos = np.zeros(info.nb, dtype=np.int32)
    _check(lib().sm_plan_export_index(plan, _np_ptr(sub_ptr), _np_ptr(sub_blocks), _np_ptr(sub_off),
                                      _np_ptr(sub_dim), _np_ptr(gen_pos)))
    return sub_ptr, sub_blocks, sub_off, sub_dim, gen_pos


def sm_sign_execute(plan, d_vals_in, mu, eps, d_vals_out, d_workspace, stats=None, stream=None) -> int:
    return _check(lib().sm_sign_execute(plan, _dev_ptr(d_vals_in), mu, eps, _dev_ptr(d_vals_out),
                                        _dev_ptr(d_workspace), d_workspace.numel() * d_workspace.element_size(),
                                        C.byref(stats) if stats is not None else None, _stream_ptr(stream)))


def sm_sign_execute_host(plan, h_vals_in, mu, eps, h_vals_out, d_workspace, stats=None, stream=None) -> int:
    """h_vals_in / h_vals_out: host numpy arrays or (pinned) CPU torch tensors."""
    pin = _dev_ptr if hasattr(h_vals_in, "data_ptr") else _np_ptr
    pout = _dev_ptr if hasattr(h_vals_out, "data_ptr") else _np_ptr
    return _check(lib().sm_sign_execute_host(plan, pin(h_vals_in), mu, eps, pout(h_vals_out),
                                             _dev_ptr(d_workspace),
                                             d_workspace.numel() * d_workspace.element_size(),
                                             C.byref(stats) if stats is not None else None, _stream_ptr(stream)))


def sm_density_matrix(plan, d_vals_in, n_target, tol_n, eps, mu0, d_vals_out, d_workspace, stats=None,
                      stream=None):
    """-> (status, mu)."""
    mu = C.c_double(mu0)
    st = _check(lib().sm_density_matrix(plan, _dev_ptr(d_vals_in), n_target, tol_n, eps, C.byref(mu),
                                        _dev_ptr(d_vals_out), _dev_ptr(d_workspace),
                                        d_workspace.numel() * d_workspace.element_size(),
                                        C.byref(stats) if stats is not None else None, _stream_ptr(stream)))
    return st, mu.value


def sm_density_matrix_host(plan, h_vals_in, n_target, tol_n, eps, mu0, h_vals_out, d_workspace, stats=None,
                           stream=None):
    mu = C.c_double(mu0)
    pin = _dev_ptr if hasattr(h_vals_in, "data_ptr") else _np_ptr
    pout = _dev_ptr if hasattr(h_vals_out, "data_ptr") else _np_ptr
    st = _check(lib().sm_density_matrix_host(plan, pin(h_vals_in), n_target, tol_n, eps, C.byref(mu),
                                             pout(h_vals_out), _dev_ptr(d_workspace),
                                             d_workspace.numel() * d_workspace.element_size(),
                                             C.byref(stats) if stats is not None else None, _stream_ptr(stream)))
    return st, mu.value


def sm_trace_dk(plan, d_D, d_K, stream=None):
    td, tdk = C.c_double(0), C.c_double(0)
    _check(lib().sm_trace_dk(plan, _dev_ptr(d_D), _dev_ptr(d_K), C.byref(td), C.byref(tdk), _stream_ptr(stream)))
    return td.value, tdk.value


SM_STATIC_MAX_NNZ = 268435456


def sm_trace_dk_static(nnz, d_D, d_K, d_out, stream=None) -> int:
    """tr(D K) into the device double d_out[0]; allocates nothing, does not synchronise (include/submatrix.h)."""
    return _check(lib().sm_trace_dk_static(int(nnz), _dev_ptr(d_D), _dev_ptr(d_K), _dev_ptr(d_out), _stream_ptr(stream)))


def sm_gather(plan, d_vals_in, mu, d_workspace, stream=None) -> int:
    return _check(lib().sm_gather(plan, _dev_ptr(d_vals_in), mu, _dev_ptr(d_workspace),
                                  d_workspace.numel() * d_workspace.element_size(), _stream_ptr(stream)))


def sm_sign_iterate(plan, eps, d_workspace, stats=None, stream=None) -> int:
    return _check(lib().sm_sign_iterate(plan, eps, _dev_ptr(d_workspace),
                                        d_workspace.numel() * d_workspace.element_size(),
                                        C.byref(stats) if stats is not None else None, _stream_ptr(stream)))


def sm_scatter(plan, as_identity, d_vals_out, d_workspace, stream=None) -> int:
    return _check(lib().sm_scatter(plan, int(as_identity), _dev_ptr(d_vals_out), _dev_ptr(d_workspace),
                                   d_workspace.numel() * d_workspace.element_size(), _stream_ptr(stream)))


def sm_set_timing(plan, enable: bool) -> int:
    return _check(lib().sm_set_timing(plan, 1 if enable else 0))


def sm_launch_count(plan) -> int:
    return int(lib().sm_launch_count(plan))


def sm_eig_decompose(plan, d_vals_in, d_workspace, stats=None, stream=None) -> int:
    return _check(lib().sm_eig_decompose(plan, _dev_ptr(d_vals_in), _dev_ptr(d_workspace),
                                         d_workspace.numel() * d_workspace.element_size(),
                                         C.byref(stats) if stats is not None else None, _stream_ptr(stream)))


def sm_eig_export(plan):
    """-> (ptr[ngroups+1], lam[sum n_i], w[sum n_i]) host copies of what Algorithm 1 keeps."""
    info = sm_plan_query(plan)
    ptr = np.zeros(info.ngroups + 1, dtype=np.int64)
    _check(lib().sm_eig_export(plan, _np_ptr(ptr), None, None))
    lam = np.zeros(int(ptr[-1]))
    w = np.zeros(int(ptr[-1]))
    _check(lib().sm_eig_export(plan, None, _np_ptr(lam), _np_ptr(w)))
    return ptr, lam, w


def sm_eig_nelec(plan, mu, kT=0.0, stream=None) -> float:
    ne = C.c_double(0)
    _check(lib().sm_eig_nelec(plan, mu, kT, C.byref(ne), _stream_ptr(stream)))
    return ne.value


def sm_eig_density(plan, mu, kT, d_vals_out, d_workspace, stream=None) -> int:
    return _check(lib().sm_eig_density(plan, mu, kT, _dev_ptr(d_vals_out), _dev_ptr(d_workspace),
                                       d_workspace.numel() * d_workspace.element_size(), _stream_ptr(stream)))


def sm_partition_groups(sub_dim, world: int) -> np.ndarray:
    """-> first[world + 1]: rank r owns groups first[r] .. first[r+1] - 1 (host only)."""
    sub_dim = np.ascontiguousarray(sub_dim, dtype=np.int32)
    first = np.zeros(world + 1, dtype=np.int32)
    _check(lib().sm_partition_groups(len(sub_dim), _np_ptr(sub_dim), world, _np_ptr(first)))
    return first


_allreduce_keepalive = {}


def make_allreduce(group=None, device=None):
    """A C callback that sums host doubles over the ranks with torch.distributed.all_reduce (plumbing:
    the tensor lives on `device`: CUDA for the nccl backend, CPU for gloo)."""
    import torch
    import torch.distributed as dist

    def _fn(ctx, vals, n):
        t = torch.tensor([vals[i] for i in range(n)], dtype=torch.float64, device=device or "cpu")
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
        out = t.cpu().tolist()
        for i in range(n):
            vals[i] = out[i]

    return ALLREDUCE_FN(_fn)


def sm_plan_set_allreduce(plan, fn) -> int:
    """fn: an ALLREDUCE_FN (make_allreduce) or None; kept alive as long as the plan uses it."""
    cb = fn if fn is not None else C.cast(None, ALLREDUCE_FN)
    _allreduce_keepalive[plan.value] = cb
    return _check(lib().sm_plan_set_allreduce(plan, cb, None))


def allgather_result(d_vals_out, info, group=None):
    """D~ of a sharded build: every rank contributes the value range of its own block columns
    (sm_plan_info_t.shard_val_begin/end) and receives the others' (plumbing over torch.distributed:
    an all-gather of unequal contiguous slices, done as broadcasts of each rank's slice)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    if info.shard_val_begin < 0:
        raise ValueError("the groups of this shard do not own one contiguous value range")
    mine = torch.tensor([info.shard_val_begin, info.shard_val_end], dtype=torch.int64, device=d_vals_out.device)
    ranges = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(ranges, mine, group=group)
    for r in range(world):
        b, e = (int(x) for x in ranges[r].tolist())
        if e > b:
            dist.broadcast(d_vals_out[b:e], src=dist.get_global_rank(group, r) if group is not None else r, group=group)
    return d_vals_out


def sm_measure_peaks(stream=None) -> sm_peaks_t:
    pk = sm_peaks_t()
    _check(lib().sm_measure_peaks(C.byref(pk), _stream_ptr(stream)))
    return pk


def sm_plan_destroy(plan) -> None:
    _allreduce_keepalive.pop(getattr(plan, "value", None), None)
    lib().sm_plan_destroy(plan)


def sm_strerror(status: int) -> str:
    return lib().sm_strerror(status).decode()


# ------------------------------------------------------------------ convenience (marshalling only)
def plan_from_matrix(m, opt=None, stream=None):
    """sm_plan_create from a workloads.BlockSparseSym."""
    return sm_plan_create(m.nb, m.blk_size, m.colptr, m.rowidx, m.ngroups, m.grp_ptr, m.grp_cols, opt, stream)


def alloc_workspace(plan, device="cuda"):
    import torch
    n = sm_plan_query(plan).workspace_bytes
    return torch.empty(max(n, 256) // 8, dtype=torch.float64, device=device)
