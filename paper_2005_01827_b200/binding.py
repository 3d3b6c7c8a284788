"""ctypes binding of libmbhl.so - argument marshalling only (include/mbhl.h is the contract).

Module-level functions carry the C names (mbhl_init, mbhl_loglike, ...) and take torch CUDA tensors
(or numpy arrays where the C call takes host pointers).  Every step of the path runs in the CUDA
library; there is no fallback: a missing library raises at import of the first call.
"""
import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmbhl.so")
NPARAM, NMODE, NQ = 11, 6, 8
COORDS_PHYSICAL, COORDS_SAMPLED, COORDS_SAMPLED_LISA = 0, 1, 2        # include/mbhl.h MBHL_COORDS_*
SYMBOLS = ("mbhl_noise", "mbhl_mode_products", "mbhl_loglike_sampled", "mbhl_loglike_coords", "mbhl_unpack_coords", "mbhl_unpack_coords_static", "mbhl_pt_init", "mbhl_pt_step", "mbhl_pt_state", "mbhl_pt_free", "mbhl_het_init", "mbhl_het_loglike", "mbhl_het_free",
           "mbhl_init", "mbhl_loglike", "mbhl_loglike_parts", "mbhl_loglike_host", "mbhl_template", "mbhl_sparse",
           "mbhl_workspace_bytes", "mbhl_set_workspace", "mbhl_data_norm", "mbhl_num_bins", "mbhl_sparse_points",
           "mbhl_launch_count", "mbhl_last_work", "mbhl_last_dense_work", "mbhl_enable_stage_timing", "mbhl_stage_times", "mbhl_dfma_probe", "mbhl_strerror", "mbhl_last_error", "mbhl_free")


class mbhl_config(ctypes.Structure):
    _fields_ = [("sparse_points", ctypes.c_int32), ("mode_mask", ctypes.c_uint32), ("t0", ctypes.c_double),
                ("max_batch", ctypes.c_int64), ("device", ctypes.c_int32), ("stream", ctypes.c_void_p)]


class MbhlError(RuntimeError):
    pass


_lib = None


def lib():
    """Loads libmbhl.so (built in-tree by paper_2005_01827_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise MbhlError(f"{LIB_PATH} not found: run `python -m paper_2005_01827_b200.build` (no CPU fallback exists)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, i32, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double
        L.mbhl_init.argtypes = [ctypes.POINTER(vp), vp, i64, vp, vp, ctypes.POINTER(mbhl_config)]
        L.mbhl_loglike.argtypes = [vp, vp, i64, vp]
        L.mbhl_loglike_parts.argtypes = [vp, vp, i64, vp, vp, vp]
        L.mbhl_loglike_host.argtypes = [vp, vp, i64, vp]
        L.mbhl_template.argtypes = [vp, vp, i64, vp, i64, vp, i32]
        L.mbhl_noise.argtypes = [vp, vp, i64, dbl, ctypes.c_uint64, vp]
        L.mbhl_mode_products.argtypes = [vp, vp, i64, vp, vp]
        L.mbhl_loglike_sampled.argtypes = [vp, vp, i64, vp]
        L.mbhl_loglike_coords.argtypes = [vp, vp, i64, i32, vp]
        L.mbhl_unpack_coords.argtypes = [vp, vp, i64, i32, vp]
        L.mbhl_unpack_coords_static.argtypes = [vp, vp, i64, i32, vp]
        L.mbhl_pt_init.argtypes = [vp, ctypes.POINTER(vp), vp, vp, i32, i32, ctypes.c_uint64, dbl, i32]
        L.mbhl_pt_step.argtypes = [vp, i32]
        L.mbhl_pt_state.argtypes = [vp, vp, vp, vp, vp]
        L.mbhl_pt_free.argtypes = [vp]
        L.mbhl_pt_free.restype = None
        L.mbhl_het_init.argtypes = [vp, ctypes.POINTER(vp), vp, vp, i32]
        L.mbhl_het_loglike.argtypes = [vp, vp, i64, vp, vp, vp]
        L.mbhl_het_free.argtypes = [vp]
        L.mbhl_het_free.restype = None
        L.mbhl_sparse.argtypes = [vp, vp, i64, vp, vp, vp]
        L.mbhl_workspace_bytes.argtypes = [vp, i64]
        L.mbhl_workspace_bytes.restype = ctypes.c_size_t
        L.mbhl_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
        L.mbhl_data_norm.argtypes = [vp]
        L.mbhl_data_norm.restype = dbl
        L.mbhl_num_bins.argtypes = [vp]
        L.mbhl_num_bins.restype = i64
        L.mbhl_sparse_points.argtypes = [vp]
        L.mbhl_sparse_points.restype = i32
        L.mbhl_launch_count.argtypes = [vp]
        L.mbhl_launch_count.restype = i64
        L.mbhl_last_work.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(i64)]
        L.mbhl_last_dense_work.argtypes = [vp, ctypes.POINTER(i64 * 5)]
        L.mbhl_enable_stage_timing.argtypes = [vp, i32]
        L.mbhl_stage_times.argtypes = [vp, ctypes.POINTER(dbl * 5)]
        L.mbhl_dfma_probe.argtypes = [vp, i32, i32, i64, vp]
        L.mbhl_strerror.argtypes = [ctypes.c_int]
        L.mbhl_strerror.restype = ctypes.c_char_p
        L.mbhl_last_error.argtypes = [vp]
        L.mbhl_last_error.restype = ctypes.c_char_p
        L.mbhl_free.argtypes = [vp]
        L.mbhl_free.restype = None
        _lib = L
    return _lib


def _check(rc, ctx=None):
    if rc != 0:
        msg = lib().mbhl_strerror(rc).decode()
        if ctx:
            msg += ": " + lib().mbhl_last_error(ctx).decode()
        raise MbhlError(f"mbhl error {rc}: {msg}")


def _ptr(x):
    """Address of a torch tensor or numpy array (contiguous float64), or None."""
    if x is None:
        return None
    if isinstance(x, torch.Tensor):
        assert x.dtype in (torch.float64, torch.complex128) and x.is_contiguous()
        return ctypes.c_void_p(x.data_ptr())
    assert x.dtype in (np.float64, np.complex128) and x.flags["C_CONTIGUOUS"]
    return ctypes.c_void_p(x.ctypes.data)


def _stream_handle(stream):
    return ctypes.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)


def mbhl_init(freqs, data_AET, psd_AET, sparse_points=1024, mode_mask=0, t0=0.0, max_batch=0, device=0, stream=None):
    """freqs [N], data_AET complex [3,N] (or float [3,N,2]), psd_AET [3,N]; numpy (host) or torch CUDA (device)."""
    cfg = mbhl_config(int(sparse_points), int(mode_mask), float(t0), int(max_batch), int(device),
                      _stream_handle(stream) if torch.cuda.is_available() else None)
    ctx = ctypes.c_void_p()
    n = int(freqs.shape[0])
    _check(lib().mbhl_init(ctypes.byref(ctx), _ptr(freqs), n, _ptr(data_AET), _ptr(psd_AET), ctypes.byref(cfg)))
    return ctx


def mbhl_free(ctx):
    lib().mbhl_free(ctx)


def mbhl_loglike(ctx, params, logL=None):
    B = int(params.shape[0])
    if logL is None:
        logL = torch.empty(B, dtype=torch.float64, device=params.device)
    _check(lib().mbhl_loglike(ctx, _ptr(params), B, _ptr(logL)), ctx)
    return logL


def mbhl_loglike_parts(ctx, params):
    B = int(params.shape[0])
    out = torch.empty((3, B), dtype=torch.float64, device=params.device)
    _check(lib().mbhl_loglike_parts(ctx, _ptr(params), B, _ptr(out[0]), _ptr(out[1]), _ptr(out[2])), ctx)
    return out[0], out[1], out[2]


def mbhl_loglike_host(ctx, params_host, logL_host):
    """params_host [B,11], logL_host [B]: host tensors/arrays (pinned for async copies); synchronous."""
    B = int(params_host.shape[0])
    _check(lib().mbhl_loglike_host(ctx, _ptr(params_host), B, _ptr(logL_host)), ctx)
    return logL_host


def mbhl_template(ctx, params, freqs_out=None, direct=False):
    B = int(params.shape[0])
    n = int(freqs_out.shape[0]) if freqs_out is not None else int(lib().mbhl_num_bins(ctx))
    out = torch.empty((B, 3, n, 2), dtype=torch.float64, device=params.device)
    _check(lib().mbhl_template(ctx, _ptr(params), B, _ptr(freqs_out), n, _ptr(out), 1 if direct else 0), ctx)
    return torch.view_as_complex(out)


def mbhl_sparse(ctx, params, want_coef=True, outputs=True):
    """Steps a1-a5 only.  outputs=False passes NULL for all three outputs (results stay in the workspace)."""
    B = int(params.shape[0])
    if not outputs:
        _check(lib().mbhl_sparse(ctx, _ptr(params), B, None, None, None), ctx)
        return None
    S = int(lib().mbhl_sparse_points(ctx))
    dev = params.device
    knots = torch.empty((B, NMODE, S), dtype=torch.float64, device=dev)
    y = torch.empty((B, NMODE, NQ, S), dtype=torch.float64, device=dev)
    coef = torch.empty((B, NMODE, S - 1, NQ, 4), dtype=torch.float64, device=dev) if want_coef else None
    _check(lib().mbhl_sparse(ctx, _ptr(params), B, _ptr(knots), _ptr(y), _ptr(coef)), ctx)
    return knots, y, coef


def mbhl_workspace_bytes(ctx, B):
    return int(lib().mbhl_workspace_bytes(ctx, int(B)))


def mbhl_set_workspace(ctx, tensor):
    if tensor is None:
        _check(lib().mbhl_set_workspace(ctx, None, 0), ctx)
    else:
        _check(lib().mbhl_set_workspace(ctx, ctypes.c_void_p(tensor.data_ptr()), tensor.numel() * tensor.element_size()), ctx)


def mbhl_data_norm(ctx):
    return float(lib().mbhl_data_norm(ctx))


def mbhl_launch_count(ctx):
    return int(lib().mbhl_launch_count(ctx))


def mbhl_last_work(ctx):
    p, b = ctypes.c_int64(), ctypes.c_int64()
    _check(lib().mbhl_last_work(ctx, ctypes.byref(p), ctypes.byref(b)), ctx)
    return p.value, b.value


def mbhl_last_dense_work(ctx):
    """(uniform calls, gated calls, per-bin-record calls, single lane evaluations, epilogues) of the last dense launch."""
    c = (ctypes.c_int64 * 5)()
    _check(lib().mbhl_last_dense_work(ctx, ctypes.byref(c)), ctx)
    return tuple(int(v) for v in c)


def mbhl_enable_stage_timing(ctx, on=True):
    _check(lib().mbhl_enable_stage_timing(ctx, 1 if on else 0), ctx)


def mbhl_stage_times(ctx):
    """Milliseconds of the last mbhl_loglike* call: (consts, sparse, spline, dense, reduce)."""
    ms = (ctypes.c_double * 5)()
    _check(lib().mbhl_stage_times(ctx, ctypes.byref(ms)), ctx)
    return list(ms)


def mbhl_dfma_probe(blocks, threads, iters, sink, stream=None):
    _check(lib().mbhl_dfma_probe(_stream_handle(stream), int(blocks), int(threads), int(iters), _ptr(sink)))


def mbhl_mode_products(ctx, params):
    """(<d|h_lm>, <h_lm|h_lm>) of every mode in isolation: two [B, 6] tensors."""
    B = int(params.shape[0])
    out = torch.empty((2, B, NMODE), dtype=torch.float64, device=params.device)
    _check(lib().mbhl_mode_products(ctx, _ptr(params), B, _ptr(out[0]), _ptr(out[1])), ctx)
    return out[0], out[1]


def mbhl_loglike_sampled(ctx, theta, logL=None):
    B = int(theta.shape[0])
    if logL is None:
        logL = torch.empty(B, dtype=torch.float64, device=theta.device)
    _check(lib().mbhl_loglike_sampled(ctx, _ptr(theta), B, _ptr(logL)), ctx)
    return logL


def mbhl_loglike_coords(ctx, rows, coords, logL=None):
    B = int(rows.shape[0])
    if logL is None:
        logL = torch.empty(B, dtype=torch.float64, device=rows.device)
    _check(lib().mbhl_loglike_coords(ctx, _ptr(rows), B, int(coords), _ptr(logL)), ctx)
    return logL


def mbhl_unpack_coords(ctx, rows, coords):
    """Physical SSB parameters [B, 11] of rows given in `coords` (NaN rows outside the prior box)."""
    B = int(rows.shape[0])
    out = torch.empty((B, NPARAM), dtype=torch.float64, device=rows.device)
    _check(lib().mbhl_unpack_coords(ctx, _ptr(rows), B, int(coords), _ptr(out)), ctx)
    return out


STATIC_MAX_WALKERS = 1024            # include/mbhl.h MBHL_STATIC_MAX_WALKERS


def mbhl_unpack_coords_static(ctx, rows, coords, out):
    """mbhl_unpack_coords for callers that must not allocate device memory (a memory pool already owns the GPU's free
    HBM, a fixed memory quota, a loop that cannot take cudaMalloc's stall): the kernel's scratch records live in a fixed
    array of the library, so the C call allocates nothing - and neither does this wrapper, which is why `out` [B, 11]
    (float64, CUDA, not overlapping `rows`) is passed in instead of created here.  At most STATIC_MAX_WALKERS rows per
    call (MbhlError above that).  Make the first call on a device during set-up; calls that can overlap on one GPU race
    on the shared array (include/mbhl.h has the full rules).  Returns `out`."""
    B = int(rows.shape[0])
    assert tuple(out.shape) == (B, NPARAM)
    _check(lib().mbhl_unpack_coords_static(ctx, _ptr(rows), B, int(coords), _ptr(out)), ctx)
    return out


def mbhl_pt_init(ctx, theta0, betas, seed=0, stretch_a=1.15, coords=COORDS_SAMPLED):
    """theta0 [T, K, 11] (torch CUDA or numpy), betas [T] numpy/host.  Returns the ensemble handle."""
    T, K = int(theta0.shape[0]), int(theta0.shape[1])
    betas = np.ascontiguousarray(betas, dtype=np.float64)
    assert betas.shape == (T,)
    pt = ctypes.c_void_p()
    _check(lib().mbhl_pt_init(ctx, ctypes.byref(pt), _ptr(theta0), _ptr(betas), T, K, ctypes.c_uint64(int(seed)), float(stretch_a), int(coords)), ctx)
    return pt


def mbhl_pt_step(pt, n_steps=1):
    _check(lib().mbhl_pt_step(pt, int(n_steps)))


def mbhl_pt_state(pt, T, K, device):
    """Returns (theta [T,K,11], logL [T,K]) as torch tensors on `device` and (n_accept [T], n_swap [T-1]) as numpy."""
    theta = torch.empty((T, K, NPARAM), dtype=torch.float64, device=device)
    logl = torch.empty((T, K), dtype=torch.float64, device=device)
    acc = np.zeros(T, dtype=np.int64)
    swp = np.zeros(max(T - 1, 1), dtype=np.int64)
    _check(lib().mbhl_pt_state(pt, _ptr(theta), _ptr(logl), ctypes.c_void_p(acc.ctypes.data), ctypes.c_void_p(swp.ctypes.data)))
    return theta, logl, acc, swp[:T - 1]


def mbhl_pt_free(pt):
    lib().mbhl_pt_free(pt)


def mbhl_noise(psd_AET, df, seed=0, stream=None):
    """Complex noise realisation [3, N] (torch CUDA complex128) for the one-sided PSD psd_AET [3, N] (torch CUDA)."""
    n = int(psd_AET.shape[1])
    out = torch.empty((3, n, 2), dtype=torch.float64, device=psd_AET.device)
    _check(lib().mbhl_noise(_stream_handle(stream), _ptr(psd_AET), n, float(df), ctypes.c_uint64(int(seed)), _ptr(out)))
    return torch.view_as_complex(out)


def mbhl_het_init(ctx, params_ref, edges):
    """Heterodyned-likelihood handle for the reference params_ref [11] (torch CUDA) and coarse-bin edges (int64 numpy, host)."""
    edges = np.ascontiguousarray(edges, dtype=np.int64)
    het = ctypes.c_void_p()
    _check(lib().mbhl_het_init(ctx, ctypes.byref(het), _ptr(params_ref), ctypes.c_void_p(edges.ctypes.data), int(edges.size - 1)), ctx)
    return het


def mbhl_het_loglike(het, params):
    """(<d|h>, <h|h>, logL) of the walkers params [B, 11] from the handle's summary data."""
    B = int(params.shape[0])
    out = torch.empty((3, B), dtype=torch.float64, device=params.device)
    _check(lib().mbhl_het_loglike(het, _ptr(params), B, _ptr(out[0]), _ptr(out[1]), _ptr(out[2])))
    return out[0], out[1], out[2]


def mbhl_het_free(het):
    lib().mbhl_het_free(het)
