"""Thin ctypes binding of the C-ABI library (include/rcg.h).  Argument marshalling only: every
step of the path runs in the CUDA kernels of librcg.so.  PyTorch supplies device memory and
streams.  There is no CPU fallback: if librcg.so is missing or no CUDA device is present the
calls raise.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("RCG_LIB") or os.path.join(_HERE, "librcg.so")   # RCG_LIB: an alternative build of the same library
_lib = None

TIER_REGISTER, TIER_WARP, TIER_GLOBAL, TIER_BLOCK = 1, 2, 3, 4
EXPORTS = ["rcg_basis_create", "rcg_basis_destroy", "rcg_eri_workspace_bytes", "rcg_eri_batch", "rcg_eri_batch_uniform",
           "rcg_eri_batch_static", "rcg_eri_batch_static_max_quartets",
           "rcg_eri_batch_host", "rcg_eri_batch_tier", "rcg_eri_workspace_bytes_tier", "rcg_validate_batch",
           "rcg_boys", "rcg_class_info", "rcg_num_classes", "rcg_class_at", "rcg_status_string",
           "rcg_last_cuda_error", "rcg_fp64_peak_tflops", "rcg_schwarz_from_blocks", "rcg_quartets_from_pairs",
           "rcg_jk_digest", "rcg_jk_finish", "rcg_fock_batch", "rcg_fock_workspace_bytes", "rcg_eri_grad_batch",
           "rcg_eri_grad_supported", "rcg_eri_grad_batch_uniform"]


class RcgError(RuntimeError):
    pass


def lib():
    """Load librcg.so (built by `python -m paper_2605_10312_b200.build`); raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RcgError("librcg.so not built: run `python -m paper_2605_10312_b200.build` (no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64
        L.rcg_basis_create.argtypes = [ctypes.POINTER(vp), i32, i32, vp, vp, vp, vp, vp, vp]
        L.rcg_basis_destroy.argtypes = [vp]
        L.rcg_eri_workspace_bytes.argtypes = [vp, i32, i32, i32, i32, i64, ctypes.POINTER(ctypes.c_size_t)]
        L.rcg_eri_workspace_bytes_tier.argtypes = [vp, i32, i32, i32, i32, i32, i64, ctypes.POINTER(ctypes.c_size_t)]
        L.rcg_eri_batch.argtypes = [vp, i32, i32, i32, i32, vp, i64, vp, vp, ctypes.c_size_t, vp]
        L.rcg_eri_batch_uniform.argtypes = [vp, i32, i32, i32, i32, vp, i64, vp, vp, ctypes.c_size_t, vp]
        L.rcg_eri_batch_static.argtypes = [vp, i32, i32, i32, i32, vp, i64, vp, vp]
        L.rcg_eri_batch_static_max_quartets.argtypes = [vp, i32, i32, i32, i32, ctypes.POINTER(i64)]
        L.rcg_eri_batch_tier.argtypes = [vp, i32, i32, i32, i32, i32, vp, i64, vp, vp, ctypes.c_size_t, vp]
        L.rcg_eri_batch_host.argtypes = [vp, i32, i32, i32, i32, vp, i64, vp, vp]
        L.rcg_eri_grad_batch.argtypes = [vp, i32, i32, i32, i32, vp, i64, vp, vp]
        L.rcg_eri_grad_batch_uniform.argtypes = [vp, i32, i32, i32, i32, vp, i64, i64, vp, vp]
        L.rcg_eri_grad_supported.argtypes = [i32, i32, i32, i32, ctypes.POINTER(i32), ctypes.POINTER(ctypes.c_size_t)]
        L.rcg_validate_batch.argtypes = [vp, i32, i32, i32, i32, vp, i64, vp]
        L.rcg_boys.argtypes = [i32, vp, i64, vp, vp]
        L.rcg_schwarz_from_blocks.argtypes = [vp, i64, i32, vp, vp]
        L.rcg_quartets_from_pairs.argtypes = [vp, vp, vp, i64, i64, vp, vp]
        L.rcg_jk_digest.argtypes = [i32, i32, i32, i32, vp, i64, vp, vp, vp, vp, vp, i32, vp]
        L.rcg_jk_finish.argtypes = [vp, vp, i32, vp]
        L.rcg_fock_workspace_bytes.argtypes = [vp, i32, i32, i32, i32, i64, i32, ctypes.POINTER(ctypes.c_size_t)]
        L.rcg_fock_batch.argtypes = [vp, i32, i32, i32, i32, vp, i64, i32, vp, vp, vp, vp, i32, vp, ctypes.c_size_t, vp]
        L.rcg_class_info.argtypes = [i32, i32, i32, i32, ctypes.POINTER(i32), ctypes.POINTER(i64), ctypes.POINTER(i64)]
        L.rcg_class_at.argtypes = [i32] + [ctypes.POINTER(i32)] * 4
        L.rcg_fp64_peak_tflops.argtypes = [ctypes.POINTER(ctypes.c_double), vp]
        L.rcg_status_string.argtypes = [i32]
        L.rcg_status_string.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _check(status):
    if status != 0:
        msg = lib().rcg_status_string(status).decode()
        if status == -4:
            msg += " (cudaError %d)" % lib().rcg_last_cuda_error()
        raise RcgError("rcg: %s" % msg)


def _stream(stream=None):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return ctypes.c_void_p(s.cuda_stream)


def nsph(l):
    return 2 * l + 1


class Basis:
    """rcg_basis handle built from the flat host arrays of workloads.make_basis."""

    def __init__(self, basis, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RcgError("no CUDA device (the library has no CPU fallback)")
        torch.cuda.init()
        torch.zeros(1, device="cuda")          # make sure the primary context is current
        self.shell_l = np.ascontiguousarray(basis["shell_l"], np.int32)
        po = np.ascontiguousarray(basis["prim_off"], np.int32)
        ex = np.ascontiguousarray(basis["exps"], np.float64)
        co = np.ascontiguousarray(basis["coefs"], np.float64)
        ce = np.ascontiguousarray(basis["centers"], np.float64)
        h = ctypes.c_void_p()
        _check(lib().rcg_basis_create(ctypes.byref(h), len(self.shell_l), len(ex), self.shell_l.ctypes.data,
                                      po.ctypes.data, ex.ctypes.data, co.ctypes.data, ce.ctypes.data, _stream(stream)))
        self.handle = h

    def close(self):
        if self.handle:
            lib().rcg_basis_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def eri_workspace_bytes(basis, lclass, nquartet, tier=0):
    n = ctypes.c_size_t()
    _check(lib().rcg_eri_workspace_bytes_tier(basis.handle, tier, *lclass, int(nquartet), ctypes.byref(n)))
    return n.value


def eri_batch(basis, lclass, quartets, out=None, workspace=None, stream=None, tier=0, uniform=False):
    """rcg_eri_batch (uniform=True: rcg_eri_batch_uniform, every quartet of the list has the same K4): quartets = CUDA int32
    tensor [n,4]; returns CUDA float64 tensor [n, 2la+1, 2lb+1, 2lc+1, 2ld+1] (asynchronous on the stream)."""
    import torch
    la, lb, lc, ld = (int(x) for x in lclass)
    assert quartets.is_cuda and quartets.dtype == torch.int32 and quartets.is_contiguous()
    n = quartets.shape[0]
    shape = (n, nsph(la), nsph(lb), nsph(lc), nsph(ld))
    if out is None:
        out = torch.empty(shape, dtype=torch.float64, device=quartets.device)
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == int(np.prod(shape))
    need = eri_workspace_bytes(basis, (la, lb, lc, ld), n, tier)
    if need and (workspace is None or workspace.numel() * workspace.element_size() < need):
        workspace = torch.empty((need + 7) // 8, dtype=torch.float64, device=quartets.device)
        if stream is not None:
            workspace.record_stream(stream)     # allocated here, used on `stream`: keep the caching allocator from reusing it early
    wsp = workspace.data_ptr() if workspace is not None else None
    wsb = workspace.numel() * workspace.element_size() if workspace is not None else 0
    if uniform and not tier:
        _check(lib().rcg_eri_batch_uniform(basis.handle, la, lb, lc, ld, quartets.data_ptr() if n else None, n,
                                           out.data_ptr() if n else None, wsp, wsb, _stream(stream)))
        return out
    _check(lib().rcg_eri_batch_tier(basis.handle, tier, la, lb, lc, ld, quartets.data_ptr() if n else None, n,
                                    out.data_ptr() if n else None, wsp, wsb, _stream(stream)))
    return out


def eri_grad_supported(lclass):
    """rcg_eri_grad_supported: (supported, shared-memory bytes of a block) for the class in the caller's order."""
    ok, sm = ctypes.c_int32(), ctypes.c_size_t()
    _check(lib().rcg_eri_grad_supported(*[int(x) for x in lclass], ctypes.byref(ok), ctypes.byref(sm)))
    return bool(ok.value), sm.value


def eri_grad_batch(basis, lclass, quartets, out=None, stream=None, k4=0):
    """rcg_eri_grad_batch: first derivatives with respect to the four centres; quartets = CUDA int32 tensor [n,4]; returns the CUDA
    float64 tensor [n, 12, 2la+1, 2lb+1, 2lc+1, 2ld+1] (derivative index 3 * column + axis), asynchronous on the stream.
    k4 > 0: rcg_eri_grad_batch_uniform (every quartet of the list has k4 primitive quartets)."""
    import torch
    la, lb, lc, ld = (int(x) for x in lclass)
    assert quartets.is_cuda and quartets.dtype == torch.int32 and quartets.is_contiguous()
    n = quartets.shape[0]
    shape = (n, 12, nsph(la), nsph(lb), nsph(lc), nsph(ld))
    if out is None:
        out = torch.empty(shape, dtype=torch.float64, device=quartets.device)
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == int(np.prod(shape))
    if k4:
        _check(lib().rcg_eri_grad_batch_uniform(basis.handle, la, lb, lc, ld, quartets.data_ptr() if n else None, n, int(k4),
                                                out.data_ptr() if n else None, _stream(stream)))
        return out
    _check(lib().rcg_eri_grad_batch(basis.handle, la, lb, lc, ld, quartets.data_ptr() if n else None, n,
                                    out.data_ptr() if n else None, _stream(stream)))
    return out


STATIC_SCRATCH_BYTES = 32 << 20


def eri_batch_static_max_quartets(basis, lclass):
    n = ctypes.c_int64()
    _check(lib().rcg_eri_batch_static_max_quartets(basis.handle, *[int(x) for x in lclass], ctypes.byref(n)))
    return n.value


def eri_batch_static(basis, lclass, quartets, out, stream=None):
    """rcg_eri_batch_static: rcg_eri_batch with the launch's scratch in the library's static device array (no allocation in the call;
    the caller passes `out`).  Only classes that use scratch; batches beyond the 32 MiB array raise."""
    import torch
    la, lb, lc, ld = (int(x) for x in lclass)
    assert quartets.is_cuda and quartets.dtype == torch.int32 and quartets.is_contiguous()
    n = quartets.shape[0]
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == n * nsph(la) * nsph(lb) * nsph(lc) * nsph(ld)
    _check(lib().rcg_eri_batch_static(basis.handle, la, lb, lc, ld, quartets.data_ptr() if n else None, n,
                                      out.data_ptr() if n else None, _stream(stream)))
    return out


def eri_batch_host(basis, lclass, quartets_host, out_host=None, stream=None):
    """rcg_eri_batch_host: numpy (or pinned torch CPU) quartets in, host integrals out; synchronous."""
    import torch
    la, lb, lc, ld = (int(x) for x in lclass)
    q = quartets_host if isinstance(quartets_host, torch.Tensor) else torch.from_numpy(
        np.ascontiguousarray(quartets_host, np.int32))
    n = q.shape[0]
    shape = (n, nsph(la), nsph(lb), nsph(lc), nsph(ld))
    if out_host is None:
        out_host = torch.empty(shape, dtype=torch.float64)
    _check(lib().rcg_eri_batch_host(basis.handle, la, lb, lc, ld, q.data_ptr(), n, out_host.data_ptr(), _stream(stream)))
    return out_host


def validate_batch(basis, lclass, quartets, stream=None):
    _check(lib().rcg_validate_batch(basis.handle, *[int(x) for x in lclass], quartets.data_ptr(), quartets.shape[0],
                                    _stream(stream)))


def schwarz_from_blocks(blocks, dim, stream=None):
    """rcg_schwarz_from_blocks: blocks = CUDA float64 [n, dim, dim] ((ab|ab) blocks); returns Q [n]."""
    import torch
    assert blocks.is_cuda and blocks.dtype == torch.float64 and blocks.is_contiguous()
    n = blocks.numel() // (dim * dim)
    Q = torch.empty(n, dtype=torch.float64, device=blocks.device)
    _check(lib().rcg_schwarz_from_blocks(blocks.data_ptr() if n else None, n, int(dim), Q.data_ptr() if n else None, _stream(stream)))
    return Q


def quartets_from_pairs(bra_pairs, ket_pairs, offs, i0, i1, nrows, out=None, stream=None):
    """rcg_quartets_from_pairs: CUDA int32 pair lists [.,2], CUDA int64 offs [nbra+1]; returns the CUDA int32
    list [nrows, 4] of bra pairs i0..i1-1 against their surviving ket prefixes (nrows = offs[i1]-offs[i0])."""
    import torch
    for t in (bra_pairs, ket_pairs):
        assert t.is_cuda and t.dtype == torch.int32 and t.is_contiguous()
    assert offs.is_cuda and offs.dtype == torch.int64 and offs.is_contiguous()
    if out is None:
        out = torch.empty((nrows, 4), dtype=torch.int32, device=bra_pairs.device)
    assert out.numel() >= 4 * nrows
    _check(lib().rcg_quartets_from_pairs(bra_pairs.data_ptr(), ket_pairs.data_ptr(), offs.data_ptr(), int(i0), int(i1),
                                         out.data_ptr() if nrows else None, _stream(stream)))
    return out[:nrows] if out.dim() == 2 else out.view(-1, 4)[:nrows]


def jk_digest(lclass, quartets, integrals, bf_off, D, Jt, Kt, stream=None):
    """rcg_jk_digest: adds the contribution of a batch of unique quartets to Jt and Kt (CUDA float64 [nbf, nbf])."""
    import torch
    n = quartets.shape[0]
    nbf = D.shape[0]
    for t in (integrals, D, Jt, Kt):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
    assert quartets.is_cuda and quartets.dtype == torch.int32 and quartets.is_contiguous()
    assert bf_off.is_cuda and bf_off.dtype == torch.int32 and D.shape == Jt.shape == Kt.shape == (nbf, nbf)
    assert integrals.numel() >= n * int(np.prod([nsph(int(l)) for l in lclass]))
    _check(lib().rcg_jk_digest(*[int(l) for l in lclass], quartets.data_ptr() if n else None, n,
                               integrals.data_ptr() if n else None, bf_off.data_ptr(), D.data_ptr(), Jt.data_ptr(),
                               Kt.data_ptr(), nbf, _stream(stream)))


def fock_workspace_bytes(basis, lclass, nquartet, uniform=False):
    n = ctypes.c_size_t()
    _check(lib().rcg_fock_workspace_bytes(basis.handle, *[int(l) for l in lclass], int(nquartet), int(bool(uniform)), ctypes.byref(n)))
    return n.value


def fock_batch(basis, lclass, quartets, bf_off, D, Jt, Kt, workspace=None, uniform=False, stream=None):
    """rcg_fock_batch: integrals of a batch of unique quartets (canonical class order) digested into Jt, Kt without storing them."""
    import torch
    n = quartets.shape[0]
    nbf = D.shape[0]
    for t in (D, Jt, Kt):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
    assert quartets.is_cuda and quartets.dtype == torch.int32 and quartets.is_contiguous()
    assert bf_off.is_cuda and bf_off.dtype == torch.int32
    need = fock_workspace_bytes(basis, lclass, n, uniform)
    if need and (workspace is None or workspace.numel() * workspace.element_size() < need):
        workspace = torch.empty((need + 7) // 8, dtype=torch.float64, device=quartets.device)
        if stream is not None:
            workspace.record_stream(stream)
    wsp = workspace.data_ptr() if workspace is not None else None
    wsb = workspace.numel() * workspace.element_size() if workspace is not None else 0
    _check(lib().rcg_fock_batch(basis.handle, *[int(l) for l in lclass], quartets.data_ptr() if n else None, n, int(bool(uniform)),
                                bf_off.data_ptr(), D.data_ptr(), Jt.data_ptr(), Kt.data_ptr(), nbf, wsp, wsb, _stream(stream)))


def jk_finish(Jt, Kt, stream=None):
    """rcg_jk_finish: Jt <- Jt + Jt^T, Kt <- Kt + Kt^T in place."""
    _check(lib().rcg_jk_finish(Jt.data_ptr(), Kt.data_ptr(), Jt.shape[0], _stream(stream)))


def boys(mmax, T, stream=None):
    """rcg_boys: T = CUDA float64 tensor [n]; returns [n, mmax+1]."""
    import torch
    assert T.is_cuda and T.dtype == torch.float64 and T.is_contiguous()
    out = torch.empty((T.shape[0], mmax + 1), dtype=torch.float64, device=T.device)
    _check(lib().rcg_boys(int(mmax), T.data_ptr(), T.shape[0], out.data_ptr(), _stream(stream)))
    return out


def class_info(lclass):
    t, fp, fq = ctypes.c_int(), ctypes.c_int64(), ctypes.c_int64()
    _check(lib().rcg_class_info(*[int(x) for x in lclass], ctypes.byref(t), ctypes.byref(fp), ctypes.byref(fq)))
    return dict(tier=t.value, flops_per_prim_quartet=fp.value, flops_per_quartet=fq.value)


def classes():
    out = []
    for i in range(lib().rcg_num_classes()):
        l = [ctypes.c_int() for _ in range(4)]
        _check(lib().rcg_class_at(i, *[ctypes.byref(x) for x in l]))
        out.append(tuple(x.value for x in l))
    return out


def fp64_peak_tflops(stream=None):
    v = ctypes.c_double()
    _check(lib().rcg_fp64_peak_tflops(ctypes.byref(v), _stream(stream)))
    return v.value
