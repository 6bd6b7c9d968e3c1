"""Thin Python binding of the C ABI in include/gwmf.h (argument marshalling only).

PyTorch is used for what the boundary leaves to the caller: the device workspace, the CUDA stream
and (in `load_segment`) pinned staging of host inputs.  Every step of the hot path runs in
libgwmf.so's kernels.  There is no fallback: if the library is missing or no CUDA device is
present, construction fails loudly.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgwmf.so")

OK, E_ARG, E_EMPTY_TEMPLATE, E_STATE, E_CAPACITY, E_CUDA, E_WORKSPACE = 0, -1, -2, -3, -4, -5, -6
PATHS = {"auto": 0, "two_pass": 1, "fused": 2, "decimated": 3}          # gwmf_path
PATH_NAMES = {v: k for k, v in PATHS.items()}

EXPORTS = [
    "gwmf_workspace_bytes", "gwmf_create", "gwmf_make_bank", "gwmf_load_segment", "gwmf_filter",
    "gwmf_filter_timed", "gwmf_triggers", "gwmf_sigma", "gwmf_effective_distance", "gwmf_trigger_distances", "gwmf_band_edges", "gwmf_transform_counts", "gwmf_series", "gwmf_correlate",
    "gwmf_fft_inverse", "gwmf_power_table_static",
    "gwmf_uses_fused", "gwmf_path_in_use", "gwmf_launch_count", "gwmf_destroy", "gwmf_strerror", "gwmf_last_cuda_error",
]


class Params(C.Structure):
    _fields_ = [("n", C.c_int64), ("fs", C.c_double), ("f_low", C.c_double), ("p", C.c_int32),
                ("rho_thresh", C.c_double), ("window", C.c_int32), ("max_templates", C.c_int32),
                ("batch", C.c_int32), ("path", C.c_int32), ("chisq_mode", C.c_int32)]


class MassPair(C.Structure):
    _fields_ = [("m1", C.c_double), ("m2", C.c_double)]


TRIGGER_DTYPE = np.dtype([("template_id", np.int32), ("sample", np.int32), ("rho", np.float32),
                          ("chisq", np.float32)])


class GwmfError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"gwmf status {status}: {text}")
        self.status = status


_lib = None


def load_library():
    """dlopen libgwmf.so (built by paper_0906_4175_b200/build.py) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(f"{LIB_PATH} not built: run `python -m paper_0906_4175_b200.build` "
                                "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.gwmf_workspace_bytes.argtypes = [C.POINTER(Params)]
    L.gwmf_workspace_bytes.restype = C.c_size_t
    L.gwmf_create.argtypes = [C.POINTER(Params), C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]
    L.gwmf_make_bank.argtypes = [C.c_void_p, C.POINTER(MassPair), C.c_int32]
    L.gwmf_load_segment.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.gwmf_filter.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
    L.gwmf_filter_timed.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_int32)]
    L.gwmf_triggers.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(C.c_int64)]
    L.gwmf_sigma.argtypes = [C.c_void_p, C.c_void_p]
    L.gwmf_band_edges.argtypes = [C.c_void_p, C.c_void_p]
    L.gwmf_effective_distance.argtypes = [C.c_void_p, C.c_double, C.c_void_p]
    L.gwmf_trigger_distances.argtypes = [C.c_void_p, C.c_double, C.c_void_p, C.c_int64, C.c_void_p]
    L.gwmf_transform_counts.argtypes = [C.c_void_p, C.c_void_p]
    L.gwmf_series.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    L.gwmf_correlate.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
    L.gwmf_fft_inverse.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.gwmf_power_table_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_double, C.c_void_p,
                                          C.c_char_p, C.c_size_t]
    L.gwmf_uses_fused.argtypes = [C.c_void_p]
    L.gwmf_path_in_use.argtypes = [C.c_void_p]
    L.gwmf_launch_count.argtypes = [C.c_void_p]
    L.gwmf_launch_count.restype = C.c_int64
    L.gwmf_destroy.argtypes = [C.c_void_p]
    L.gwmf_destroy.restype = None
    L.gwmf_strerror.argtypes = [C.c_int]
    L.gwmf_strerror.restype = C.c_char_p
    L.gwmf_last_cuda_error.argtypes = [C.c_void_p]
    L.gwmf_last_cuda_error.restype = C.c_char_p
    _lib = L
    return L


def workspace_bytes(n, p, window, max_templates, fs=4096.0, f_low=40.0, rho_thresh=6.0, batch=0, path="auto",
                    chisq_on_demand=False) -> int:
    prm = Params(int(n), float(fs), float(f_low), int(p), float(rho_thresh), int(window), int(max_templates), int(batch),
                 PATHS[path], 1 if chisq_on_demand else 0)
    return int(load_library().gwmf_workspace_bytes(C.byref(prm)))


STATIC_MAX_N = 1 << 22            # GWMF_STATIC_MAX_N


def power_table_static(Sn, n, fs=4096.0, f_low=40.0, out=None, stream=None):
    """gwmf_power_table_static: the Eq. 4 power table C[k] (n/2 fp64 entries) of the PSD `Sn`, computed without a
    context or a workspace and without any device allocation inside the library (its scratch is a static array in the
    library image) -- for callers that must not cudaMalloc when the PSD changes; see include/gwmf.h.

    Sn: torch float64 CUDA tensor of n/2 + 1 samples.  out: optional torch float64 CUDA tensor of n/2 entries on the
    same device (pass one to keep this wrapper allocation-free too; otherwise it is created here, which is the
    wrapper's doing, not the library's).  The work runs on `stream` (default: torch's current stream of Sn's device)
    and the call returns when it is done.  Calls that may overlap on one GPU must be serialised by the caller."""
    import torch
    L = load_library()
    if not (isinstance(Sn, torch.Tensor) and Sn.is_cuda and Sn.dtype == torch.float64 and Sn.is_contiguous()):
        raise TypeError("Sn must be a contiguous float64 CUDA tensor")
    if Sn.numel() != int(n) // 2 + 1:
        raise ValueError("Sn must hold n/2 + 1 samples")
    if out is None:
        out = torch.empty(int(n) // 2, dtype=torch.float64, device=Sn.device)
    if not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == int(n) // 2
            and out.device == Sn.device):
        raise TypeError("out must be a contiguous float64 CUDA tensor of n/2 entries on Sn's device")
    err = C.create_string_buffer(256)
    with torch.cuda.device(Sn.device):
        st = stream if stream is not None else torch.cuda.current_stream(Sn.device)
        rc = L.gwmf_power_table_static(C.c_void_p(Sn.data_ptr()), C.c_void_p(out.data_ptr()), int(n), float(fs),
                                       float(f_low), C.c_void_p(st.cuda_stream), err, len(err))
    if rc != OK:
        raise GwmfError(rc, err.value.decode() or L.gwmf_strerror(rc).decode())
    return out


class Filter:
    """One gwmf context: a device workspace, a stream, a bank and the current segment."""

    def __init__(self, n, p, window, max_templates, rho_thresh=6.0, fs=4096.0, f_low=40.0, batch=0,
                 device="cuda:0", stream=None, path="auto", chisq_on_demand=False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("gwmf needs a CUDA device (sm_100a); there is no CPU fallback")
        self._L = load_library()
        self.torch = torch
        self.device = torch.device(device)
        self.n, self.p, self.window = int(n), int(p), int(window)
        self.params = Params(int(n), float(fs), float(f_low), int(p), float(rho_thresh), int(window),
                             int(max_templates), int(batch), PATHS[path], 1 if chisq_on_demand else 0)
        nbytes = int(self._L.gwmf_workspace_bytes(C.byref(self.params)))
        if nbytes == 0:
            raise GwmfError(E_ARG, "invalid parameters")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) // 256 * 256
            h = C.c_void_p()
            rc = self._L.gwmf_create(C.byref(self.params), C.c_void_p(self._ws_ptr), C.c_size_t(nbytes),
                                     C.c_void_p(self.stream.cuda_stream), C.byref(h))
        self._h = h if rc == OK else None
        self._check(rc)
        self.workspace_nbytes = nbytes
        self.n_templates = 0
        self._pin_s = None
        self._pin_sn = None

    # ------------------------------------------------------------------ plumbing
    def _check(self, rc):
        if rc != OK:
            text = self._L.gwmf_strerror(rc).decode()
            if rc == E_CUDA and self._h is not None:
                text += ": " + self._L.gwmf_last_cuda_error(self._h).decode()
            raise GwmfError(rc, text)

    def close(self):
        if getattr(self, "_h", None) is not None:
            self._L.gwmf_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def synchronize(self):
        self.stream.synchronize()

    @property
    def launch_count(self) -> int:
        return int(self._L.gwmf_launch_count(self._h))

    # ------------------------------------------------------------------ the four calls of the boundary
    @property
    def uses_fused(self) -> bool:
        return bool(self._L.gwmf_uses_fused(self._h))

    @property
    def path(self) -> str:
        """The path the library resolved at create: two_pass, fused or decimated."""
        return PATH_NAMES[int(self._L.gwmf_path_in_use(self._h))]

    def make_bank(self, masses):
        arr = (MassPair * len(masses))(*[MassPair(float(a), float(b)) for a, b in masses])
        self._check(self._L.gwmf_make_bank(self._h, arr, len(masses)))
        self.n_templates = len(masses)

    def load_segment(self, s, Sn=None):
        """s: n samples (numpy or torch, host or device; cast to fp32); Sn: n/2+1 PSD samples (fp64), or None to keep
        the PSD of the previous call (then a host segment is uploaded and prepared beside the running filters)."""
        torch = self.torch
        keep = []

        def as_ptr(x, dtype):
            if isinstance(x, torch.Tensor):
                t = x.to(dtype).contiguous()
                keep.append(t)
                return t.data_ptr()
            a = np.ascontiguousarray(x, dtype=np.float32 if dtype == torch.float32 else np.float64)
            keep.append(a)
            return a.ctypes.data

        ps = as_ptr(s, torch.float32)
        pn = as_ptr(Sn, torch.float64) if Sn is not None else None
        self._check(self._L.gwmf_load_segment(self._h, C.c_void_p(ps), C.c_void_p(pn)))
        # device sources are read asynchronously on the stream: keep them alive until it drains
        if any(isinstance(k, torch.Tensor) and k.is_cuda for k in keep):
            self._keepalive = keep

    def filter(self, first=0, count=None):
        if count is None:
            count = self.n_templates - first
        self._check(self._L.gwmf_filter(self._h, int(first), int(count)))

    def filter_timed(self, first=0, count=None):
        """As filter(), returning ((ms_spectra, ms_pass1, ms_pass2, ms_chisq_at_events), (launches timed in each)); syncs."""
        if count is None:
            count = self.n_templates - first
        ms = (C.c_double * 4)()
        nl = (C.c_int32 * 4)()
        self._check(self._L.gwmf_filter_timed(self._h, int(first), int(count), ms, nl))
        return tuple(ms), tuple(nl)

    def triggers(self, capacity=None) -> np.ndarray:
        if capacity is None:
            capacity = max(1, self.n_templates) * (self.n // self.window)
        out = np.zeros(capacity, dtype=TRIGGER_DTYPE)
        n_out = C.c_int64(0)
        rc = self._L.gwmf_triggers(self._h, out.ctypes.data_as(C.c_void_p), int(capacity), C.byref(n_out))
        if rc == E_CAPACITY:
            raise GwmfError(rc, f"need capacity {n_out.value}")
        self._check(rc)
        return out[: n_out.value]

    # ------------------------------------------------------------------ parity / debug entries
    def sigma(self) -> np.ndarray:
        out = np.zeros(self.n_templates, dtype=np.float64)
        self._check(self._L.gwmf_sigma(self._h, out.ctypes.data_as(C.c_void_p)))
        return out

    def effective_distance(self, psd_unit=9e-46) -> np.ndarray:
        """Mpc at which each template has optimal SNR 1 in the loaded PSD (psd_unit: strain^2/Hz per unit of S_n)."""
        out = np.zeros(self.n_templates, dtype=np.float64)
        self._check(self._L.gwmf_effective_distance(self._h, float(psd_unit), out.ctypes.data_as(C.c_void_p)))
        return out

    def trigger_distances(self, triggers, psd_unit=9e-46) -> np.ndarray:
        """Effective distance in Mpc of each event of a Filter.triggers() array."""
        trig = np.ascontiguousarray(triggers, dtype=TRIGGER_DTYPE)
        out = np.zeros(len(trig), dtype=np.float64)
        self._check(self._L.gwmf_trigger_distances(self._h, float(psd_unit), trig.ctypes.data_as(C.c_void_p), len(trig),
                                                   out.ctypes.data_as(C.c_void_p)))
        return out

    def band_edges(self) -> np.ndarray:
        out = np.zeros((self.n_templates, self.p + 1), dtype=np.int32)
        self._check(self._L.gwmf_band_edges(self._h, out.ctypes.data_as(C.c_void_p)))
        return out

    def transform_counts(self) -> np.ndarray:
        """n-point transforms the library runs per template with its path (bench.py's byte model)."""
        out = np.zeros(self.n_templates, dtype=np.int32)
        self._check(self._L.gwmf_transform_counts(self._h, out.ctypes.data_as(C.c_void_p)))
        return out

    def series(self, template_id):
        rho = np.empty(self.n, dtype=np.float32)
        chi = np.empty(self.n, dtype=np.float32)
        self._check(self._L.gwmf_series(self._h, int(template_id), rho.ctypes.data_as(C.c_void_p),
                                        chi.ctypes.data_as(C.c_void_p)))
        return rho, chi

    def correlate(self, template_id) -> np.ndarray:
        q = np.empty(self.n // 2, dtype=np.complex64)
        self._check(self._L.gwmf_correlate(self._h, int(template_id), q.ctypes.data_as(C.c_void_p)))
        return q

    def fft_inverse(self, x):
        """x: torch complex64 device tensor of n points -> unnormalised e^{+2 pi i jk/n} transform."""
        torch = self.torch
        assert x.is_cuda and x.dtype == torch.complex64 and x.numel() == self.n
        xin = torch.view_as_real(x.contiguous())
        out = torch.empty_like(xin)
        self._check(self._L.gwmf_fft_inverse(self._h, C.c_void_p(xin.data_ptr()), C.c_void_p(out.data_ptr())))
        self._keepalive = (xin, out)
        return torch.view_as_complex(out)
