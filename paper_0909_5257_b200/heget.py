"""Thin Python binding of the C-ABI in include/heget.h: argument marshalling only.

Every step of the hot path (Philox + RAMBO + cuts, wavefunctions, vertex chain, colour form, helicity sum; eq. 4 of the
paper) runs in the CUDA kernels behind `libheget.so`.  PyTorch is used here for device memory and streams
only.  There is no CPU fallback: if the library is not built the import of a `Process` raises.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libheget.so")

OK, EINVAL, EUNSUPPORTED, ECUDA, ENOMEM, ECOMPILE = range(6)
FP64, FP32, FP32X2 = 0, 1, 2
HEL_SUM, HEL_SAMPLE, HEL_FIXED = 0, 1, 2

KERNEL_AUTO, KERNEL_STRAIGHT, KERNEL_TABLE = 0, 1, 2

EXPORTS = ["heget_process_create", "heget_process_info", "heget_color_matrix", "heget_sample_momenta", "heget_eval_me2",
           "heget_run_host", "heget_set_lanes", "heget_set_kernel", "heget_set_colour_stage", "heget_fma_probe", "heget_destroy", "heget_last_error", "heget_launch_count",
           "heget_static_prepare", "heget_static_max_events", "heget_eval_me2_static"]


class HegetError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("heget status %d: %s" % (status, message))
        self.status = status


class Cuts(C.Structure):
    _fields_ = [("pt_min", C.c_double), ("eta_max", C.c_double), ("dr_min", C.c_double)]


class Info(C.Structure):
    _fields_ = [("n_ext", C.c_int), ("n_hel", C.c_int), ("n_hel_eval", C.c_int), ("n_diagrams", C.c_int),
                ("n_topologies", C.c_int), ("n_color", C.c_int), ("n_color_eval", C.c_int), ("n_color_reduced", C.c_int), ("n_color_accum", C.c_int), ("color_rank", C.c_int),
                ("avg_spin", C.c_double), ("avg_color", C.c_double), ("sym_factor", C.c_double),
                ("flops_per_event", C.c_double), ("flops_per_helicity", C.c_double),
                ("regs_per_thread", C.c_int), ("local_bytes_per_thread", C.c_int), ("threads_per_block", C.c_int), ("lanes_wide", C.c_int), ("lanes", C.c_int),
                ("kernel", C.c_int), ("events_per_block", C.c_int), ("n_hel_computed", C.c_int), ("colour_stage", C.c_int), ("n_color_distinct", C.c_int), ("packed_pairs", C.c_int), ("j_in_tmem", C.c_int), ("flops_per_event_tensor", C.c_double), ("warps_per_j", C.c_int)]


_lib = None


def lib():
    """Load libheget.so (built in-tree by paper_0909_5257_b200/build.py); fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s is not built: run `python -m paper_0909_5257_b200.build` (no CPU fallback exists)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp, u64 = C.c_void_p, C.c_uint64
        L.heget_last_error.restype = C.c_char_p
        L.heget_launch_count.restype = u64
        L.heget_process_create.argtypes = [C.c_char_p, C.c_double, C.c_double, C.POINTER(Cuts), C.c_int, C.POINTER(vp)]
        L.heget_process_info.argtypes = [vp, C.POINTER(Info)]
        L.heget_color_matrix.argtypes = [vp, C.c_int, vp, C.POINTER(C.c_int)]
        L.heget_sample_momenta.argtypes = [vp, u64, u64, u64, vp, vp, vp, vp]
        L.heget_eval_me2.argtypes = [vp, vp, u64, C.c_int, vp, u64, u64, vp, vp]
        L.heget_run_host.argtypes = [vp, u64, u64, u64, vp, vp, vp, C.c_int, vp, vp, vp]
        L.heget_set_lanes.argtypes = [vp, C.c_int]
        L.heget_set_kernel.argtypes = [vp, C.c_int]
        L.heget_set_colour_stage.argtypes = [vp, C.c_int]
        L.heget_fma_probe.argtypes = [C.c_int, u64, vp, u64, C.POINTER(C.c_double), vp]
        L.heget_destroy.argtypes = [vp]
        L.heget_static_prepare.argtypes = [vp]
        L.heget_static_max_events.argtypes = [vp]
        L.heget_static_max_events.restype = u64
        L.heget_eval_me2_static.argtypes = [vp, vp, u64, vp, vp]
        L.heget_destroy.restype = None
        _lib = L
    return _lib


def launch_count():
    return int(lib().heget_launch_count())


def _check(st):
    if st != OK:
        raise HegetError(st, lib().heget_last_error().decode())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _dptr(t, dtype, numel, name):
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous() and t.numel() == numel):
        raise ValueError("%s must be a contiguous CUDA tensor of dtype %s with %d elements" % (name, dtype, numel))
    return C.c_void_p(t.data_ptr())


def _hptr(t, dtype, numel, name):
    if t is None:
        return None
    if not ((not t.is_cuda) and t.dtype == dtype and t.is_contiguous() and t.numel() == numel):
        raise ValueError("%s must be a contiguous host tensor of dtype %s with %d elements" % (name, dtype, numel))
    return C.c_void_p(t.data_ptr())


class Process:
    """heget_process_create / heget_destroy.  `precision` is "fp64", "fp32" or "fp32x2" (FP32 on packed f32x2 instructions)."""

    def __init__(self, process, sqrt_s_hat, alpha_s=0.118, cuts=(20.0, 2.5, 0.4), precision="fp64", kernel=None):
        self._h = None
        self.precision = {"fp64": FP64, "fp32": FP32, "fp32x2": FP32X2}[precision]
        self.dtype = torch.float64 if self.precision == FP64 else torch.float32
        c = Cuts(*cuts) if cuts is not None else None
        h = C.c_void_p()
        _check(lib().heget_process_create(process.encode(), float(sqrt_s_hat), float(alpha_s),
                                          C.byref(c) if c is not None else None, self.precision, C.byref(h)))
        self._h = h
        self.process, self.sqrt_s_hat, self.alpha_s = process, float(sqrt_s_hat), float(alpha_s)
        if kernel is not None:
            _check(lib().heget_set_kernel(self._h, {"auto": KERNEL_AUTO, "straight": KERNEL_STRAIGHT, "table": KERNEL_TABLE}[kernel]))
        self.info = self.process_info()
        self.n_ext = self.info.n_ext

    def close(self):
        if self._h is not None:
            lib().heget_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def process_info(self):
        i = Info()
        _check(lib().heget_process_info(self._h, C.byref(i)))
        return i

    def color_matrix(self, which=0):
        n = C.c_int()
        _check(lib().heget_color_matrix(self._h, which, None, C.byref(n)))
        m = torch.zeros(n.value, n.value, dtype=torch.float64)
        _check(lib().heget_color_matrix(self._h, which, C.c_void_p(m.data_ptr()), C.byref(n)))
        return m

    def set_kernel(self, kernel):
        """heget_set_kernel: "auto", "straight" (specialised compiled kernel) or "table" (generic table-driven kernels)."""
        _check(lib().heget_set_kernel(self._h, {"auto": KERNEL_AUTO, "straight": KERNEL_STRAIGHT, "table": KERNEL_TABLE}[kernel]))
        self.info = self.process_info()

    def set_colour_stage(self, stage):
        """heget_set_colour_stage: "symmetric", "distinct" (the paper's value table + index map), "cholesky" or "tensor" (tensor-core contraction through HBM); TABLE back end."""
        _check(lib().heget_set_colour_stage(self._h, {"symmetric": 0, "distinct": 1, "cholesky": 2, "tensor": 3}[stage]))
        self.info = self.process_info()

    def set_lanes(self, lanes):
        _check(lib().heget_set_lanes(self._h, int(lanes)))
        self.info = self.process_info()

    def sample_momenta(self, seed, n_events, first_event=0, mom=None, weight=None, tries=None, stream=None):
        """heget_sample_momenta: fills (and returns) mom[n_ext,4,E] float64, weight[E] float64, tries[E] int32 (uint32 bits)."""
        dev = torch.device("cuda", torch.cuda.current_device())
        if mom is None:
            mom = torch.empty(self.n_ext, 4, n_events, dtype=torch.float64, device=dev)
        _check(lib().heget_sample_momenta(self._h, seed, first_event, n_events,
                                          _dptr(mom, torch.float64, self.n_ext * 4 * n_events, "mom"),
                                          _dptr(weight, torch.float64, n_events, "weight"),
                                          _dptr(tries, torch.int32, n_events, "tries"), _stream(stream)))
        return mom

    def eval_me2(self, mom, mode=HEL_SUM, hel=None, seed=0, first_event=0, out=None, stream=None):
        """heget_eval_me2 on device momenta mom[n_ext,4,E]; returns me2[E] (float64 or float32 per the handle)."""
        n_events = mom.numel() // (self.n_ext * 4)
        if out is None:
            out = torch.empty(n_events, dtype=self.dtype, device=mom.device)
        helbuf = (C.c_int8 * self.n_ext)(*[int(x) for x in hel]) if hel is not None else None
        _check(lib().heget_eval_me2(self._h, _dptr(mom, torch.float64, self.n_ext * 4 * n_events, "mom"), n_events, mode,
                                    helbuf, seed, first_event, _dptr(out, self.dtype, n_events, "out"), _stream(stream)))
        return out

    def static_prepare(self):
        """heget_static_prepare: set-up of the entry point that allocates nothing (TABLE back end + tensor colour stage selected before)."""
        _check(lib().heget_static_prepare(self._h))

    @property
    def static_max_events(self):
        """heget_static_max_events: events one eval_me2_static call takes (0: not prepared)."""
        return int(lib().heget_static_max_events(self._h))

    def eval_me2_static(self, mom, out, stream=None):
        """heget_eval_me2_static: HEL_SUM on device momenta mom[n_ext,4,E] into the caller's out[E]; no allocation anywhere in the call."""
        n_events = mom.numel() // (self.n_ext * 4)
        _check(lib().heget_eval_me2_static(self._h, _dptr(mom, torch.float64, self.n_ext * 4 * n_events, "mom"), n_events,
                                           _dptr(out, self.dtype, n_events, "out"), _stream(stream)))
        return out

    def run_host(self, seed, n_events, first_event=0, mom_in=None, mom_out=None, weight=None, mode=HEL_SUM, hel=None,
                 out=None, stream=None):
        """heget_run_host: HOST tensors in/out; copies and kernels on `stream`, synchronised on return."""
        if out is None:
            out = torch.empty(n_events, dtype=self.dtype)
        nm = self.n_ext * 4 * n_events
        helbuf = (C.c_int8 * self.n_ext)(*[int(x) for x in hel]) if hel is not None else None
        _check(lib().heget_run_host(self._h, seed, first_event, n_events, _hptr(mom_in, torch.float64, nm, "mom_in"),
                                    _hptr(mom_out, torch.float64, nm, "mom_out"), _hptr(weight, torch.float64, n_events, "weight"),
                                    mode, helbuf, _hptr(out, self.dtype, n_events, "out"), _stream(stream)))
        return out


def fma_probe(precision, iters, n_threads, stream=None):
    """heget_fma_probe: enqueue the FMA-chain microbenchmark; returns the flops it performs."""
    dt = torch.float64 if precision == FP64 else torch.float32
    out = torch.empty(n_threads, dtype=dt, device="cuda")
    fl = C.c_double()
    _check(lib().heget_fma_probe(precision, iters, C.c_void_p(out.data_ptr()), n_threads, C.byref(fl), _stream(stream)))
    return fl.value


def shard_range(n_events, rank, world_size):
    """8(e): rank r of R takes global events [r E/R, (r+1) E/R) -- (first_event, count); no collective on the path."""
    lo = (n_events * rank) // world_size
    hi = (n_events * (rank + 1)) // world_size
    return lo, hi - lo
