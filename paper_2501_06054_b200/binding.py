"""ctypes binding of include/sas.h -- argument marshalling only.

PyTorch appears here for device memory (histograms, dump buffers) and the CUDA stream handed to
the library; nothing is computed in Python or torch.  The library must be present: a missing or
unloadable libsas_b200.so raises, it is never replaced by another path.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libsas_b200.so")

EXPORTED_SYMBOLS = [
    "sas_create_instrument", "sas_bind_buffers", "sas_set_model", "sas_trace", "sas_trace_range",
    "sas_trace_dump", "sas_read_detector", "sas_get_counters", "sas_reset_detector", "sas_destroy",
    "sas_last_error", "sas_create_batch", "sas_trace_batch", "sas_quadrature_nodes",
    "sas_get_launch_info", "sas_get_kernel_time", "sas_get_upload_bytes", "sas_version", "sas_reduce_radial",
    "sas_trace_batch_range", "sas_get_launch_records", "sas_get_reduce_time", "sas_set_launch_timing",
    "sas_reduce_radial_static",
]

SAMPLE = {"box": 0, "cyl_y": 1}
LAMBDA_DIST = {"uniform": 0, "triangle": 1}
MODEL = {"sphere": 0, "core_shell_sphere": 1, "cylinder": 2, "triaxial": 3, "core_shell_triaxial": 4, "flat": 5,
         "parallelepiped": 6, "core_shell_cylinder": 7, "ellipsoid": 8, "barbell": 9, "capped_cylinder": 10,
         "elliptical_cylinder": 11, "hollow_cylinder": 12, "core_shell_ellipsoid": 13, "polymer_micelle": 14,
         "hollow_prism_thin": 15}
ORIENT = {"fixed": 0, "gauss_quad": 1, "isotropic_mc": 2, "uniform_angles_mc": 3}
PD = {"none": 0, "schulz": 1, "gauss_mc": 2}
SQ = {"none": 0, "hard_sphere_py": 1, "hayter_msa": 2}
PRECISION = {"fp32": 0, "fp64": 1}
STATUS = {0: "SAS_OK", 1: "SAS_EINVAL", 2: "SAS_ESTATE", 3: "SAS_ECUDA", 4: "SAS_ENOMEM", 5: "SAS_EUNSUPPORTED"}


class SasError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class InstrumentDesc(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("sample_shape", C.c_int32)] + \
               [(n, C.c_double) for n in
                ("src_xw", "src_yh", "lambda_min", "lambda_max", "flux",
                 "slit1_z", "slit1_xw", "slit1_yh", "slit2_z", "slit2_xw", "slit2_yh",
                 "focus_z", "focus_xw", "focus_yh", "sample_z", "sample_xw", "sample_yh", "sample_zd",
                 "sample_radius", "mu_abs_2200", "mu_inc", "q_min", "q_max", "det_dist", "det_xw", "det_yh")] + \
               [("det_nx", C.c_int32), ("det_ny", C.c_int32), ("lambda_dist", C.c_int32), ("reserved", C.c_int32)]


class ModelDesc(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("model", C.c_int32), ("precision", C.c_int32),
                ("orient_kind", C.c_int32), ("sq_kind", C.c_int32), ("pd_kind", C.c_int32 * 2),
                ("pd_nodes", C.c_int32 * 2), ("n_theta", C.c_int32), ("n_phi", C.c_int32),
                ("reserved", C.c_int32), ("scale", C.c_double), ("background", C.c_double),
                ("sld", C.c_double * 3), ("size", C.c_double * 4), ("pd_rel", C.c_double * 2),
                ("theta", C.c_double), ("phi", C.c_double), ("psi", C.c_double),
                ("sigma_theta", C.c_double), ("sigma_phi", C.c_double),
                ("sq_radius_eff", C.c_double), ("sq_volfrac", C.c_double),
                ("sq_contact_kT", C.c_double), ("sq_kappa_sigma", C.c_double)]


class RadialDesc(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("exp_index", C.c_uint32), ("n_bins", C.c_int32), ("reserved", C.c_int32),
                ("q_lo", C.c_double), ("q_hi", C.c_double), ("lambda_ref", C.c_double), ("n_launched", C.c_uint64)]


class LaunchRecord(C.Structure):
    _fields_ = [("variant", C.c_int32), ("per_event", C.c_int32), ("precision", C.c_int32),
                ("warp_specialised", C.c_int32), ("n_exp", C.c_uint32), ("n_per_exp", C.c_uint32),
                ("grid", C.c_int32), ("block", C.c_int32), ("ms", C.c_double)]


MAX_LAUNCH_RECORDS = 4096


def instrument_desc(d: dict) -> InstrumentDesc:
    s = InstrumentDesc()
    s.struct_size = C.sizeof(InstrumentDesc)
    for name, typ in InstrumentDesc._fields_:
        if name == "struct_size":
            continue
        if name == "reserved":
            continue
        if name == "lambda_dist":
            v = d.get(name, "uniform")
            s.lambda_dist = LAMBDA_DIST[v] if isinstance(v, str) else int(v)
        elif name == "sample_shape":
            s.sample_shape = SAMPLE[d[name]] if isinstance(d[name], str) else int(d[name])
        elif typ is C.c_int32:
            setattr(s, name, int(d[name]))
        else:
            setattr(s, name, float(d[name]))
    return s


def model_desc(d: dict) -> ModelDesc:
    as_int = lambda table, v: table[v] if isinstance(v, str) else int(v)
    m = ModelDesc()
    m.struct_size = C.sizeof(ModelDesc)
    m.model = as_int(MODEL, d["model"])
    m.precision = as_int(PRECISION, d["precision"])
    m.orient_kind = as_int(ORIENT, d["orient_kind"])
    m.sq_kind = as_int(SQ, d["sq_kind"])
    for k in range(2):
        m.pd_kind[k] = as_int(PD, d["pd_kind"][k])
        m.pd_nodes[k] = int(d["pd_nodes"][k])
        m.pd_rel[k] = float(d["pd_rel"][k])
    m.n_theta, m.n_phi = int(d["n_theta"]), int(d["n_phi"])
    m.scale, m.background = float(d["scale"]), float(d["background"])
    for i in range(3):
        m.sld[i] = float(d["sld"][i])
    for i in range(4):
        m.size[i] = float(d["size"][i])
    m.theta, m.phi, m.psi = float(d["theta"]), float(d["phi"]), float(d["psi"])
    m.sigma_theta, m.sigma_phi = float(d["sigma_theta"]), float(d["sigma_phi"])
    m.sq_radius_eff, m.sq_volfrac = float(d["sq_radius_eff"]), float(d["sq_volfrac"])
    m.sq_contact_kT, m.sq_kappa_sigma = float(d.get("sq_contact_kT", 0.0)), float(d.get("sq_kappa_sigma", 0.0))
    return m


_lib = None


def load_library(path: str | None = None):
    """Load libsas_b200.so and declare the prototypes. Raises if the library is absent."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or _LIB_PATH
    if not os.path.exists(p):
        raise FileNotFoundError(
            f"{p} is missing: build it with `python -m paper_2501_06054_b200.build` "
            "(there is no CPU fallback for the CUDA path)")
    L = C.CDLL(p)
    vp, u64, u32, i32, dbl = C.c_void_p, C.c_uint64, C.c_uint32, C.c_int32, C.c_double
    pp = C.POINTER
    L.sas_create_instrument.argtypes = [pp(InstrumentDesc), pp(vp)]
    L.sas_bind_buffers.argtypes = [vp, vp, vp, vp, vp]
    L.sas_set_model.argtypes = [vp, pp(ModelDesc)]
    L.sas_trace.argtypes = [vp, u64, u64]
    L.sas_trace_range.argtypes = [vp, u64, u64, u64]
    L.sas_trace_dump.argtypes = [vp, u64, u64, u64, u32, vp, vp, vp]
    L.sas_read_detector.argtypes = [vp, vp, vp, vp]
    L.sas_get_counters.argtypes = [vp, pp(u64)]
    L.sas_reset_detector.argtypes = [vp]
    L.sas_destroy.argtypes = [vp]
    L.sas_destroy.restype = None
    L.sas_last_error.argtypes = [vp]
    L.sas_last_error.restype = C.c_char_p
    L.sas_create_batch.argtypes = [pp(InstrumentDesc), pp(ModelDesc), u32, pp(vp)]
    L.sas_trace_batch.argtypes = [vp, u64, u64]
    L.sas_trace_batch_range.argtypes = [vp, u64, u64, u64]
    L.sas_get_launch_records.argtypes = [vp, pp(LaunchRecord), u32, pp(u32)]
    L.sas_get_reduce_time.argtypes = [vp, pp(dbl)]
    L.sas_quadrature_nodes.argtypes = [i32, dbl, i32, pp(dbl), pp(dbl)]
    L.sas_get_launch_info.argtypes = [vp, pp(u64), pp(i32), pp(i32), pp(i32)]
    L.sas_get_kernel_time.argtypes = [vp, i32, pp(dbl), pp(u64)]
    L.sas_set_launch_timing.argtypes = [vp, i32]
    L.sas_get_upload_bytes.argtypes = [vp, pp(u64)]
    L.sas_reduce_radial.argtypes = [vp, pp(RadialDesc), vp, vp, vp, vp]
    L.sas_reduce_radial_static.argtypes = [pp(InstrumentDesc), pp(RadialDesc), vp, vp, vp, vp, vp, vp, vp]
    L.sas_version.argtypes = []
    L.sas_version.restype = C.c_char_p
    for name in EXPORTED_SYMBOLS:
        if name not in ("sas_destroy", "sas_last_error", "sas_version"):
            getattr(L, name).restype = C.c_int
    if path is None:
        _lib = L
    return L


def _check(L, ctx, status):
    if status != 0:
        raise SasError(status, (L.sas_last_error(ctx) or b"").decode())


def quadrature_nodes(kind: str, param: float, n: int):
    """Host-only: the rule the library uses ('schulz' | 'gauss_tilt'). Returns (values, weights)."""
    L = load_library()
    v = (C.c_double * n)()
    w = (C.c_double * n)()
    _check(L, None, L.sas_quadrature_nodes({"schulz": 0, "gauss_tilt": 1}[kind], float(param), n, v, w))
    return np.array(v[:]), np.array(w[:])


def reduce_radial_static(instrument: dict, sum_p, sum_p2, n_launched, lambda_ref, q_lo, q_hi, n_bins, out=None, stream=None):
    """sas_reduce_radial_static (include/sas.h): ring average of one detector image without any allocation inside
    the library.  sum_p, sum_p2: CUDA float64 tensors [ny][nx]; out: four caller-owned CUDA tensors (q, I, sigma
    float64, npix int64/uint64 storage) of n_bins entries -- made here when omitted (by torch, outside the library).
    Asynchronous on `stream` (default: torch's current stream of the inputs' device); returns `out`."""
    import torch
    L = load_library()
    ins = instrument_desc(instrument)
    d = RadialDesc(C.sizeof(RadialDesc), 0, int(n_bins), 0, float(q_lo), float(q_hi), float(lambda_ref), int(n_launched))
    dev = sum_p.device
    if out is None:
        out = tuple(torch.empty(max(int(n_bins), 1), dtype=dt, device=dev) for dt in (torch.float64, torch.float64, torch.float64, torch.int64))
    with torch.cuda.device(dev):
        st = (stream if stream is not None else torch.cuda.current_stream(dev)).cuda_stream
        _check(L, None, L.sas_reduce_radial_static(C.byref(ins), C.byref(d), sum_p.data_ptr(), sum_p2.data_ptr(),
                                                   *(t.data_ptr() for t in out), st))
    return out


class _Base:
    """Owns a sas_ctx plus torch-allocated device histograms bound to it."""

    @staticmethod
    def _device(device):
        """torch.device of the context: the given one, else torch's current CUDA device."""
        import torch
        if not torch.cuda.is_available():
            raise SasError(3, "no CUDA device: the tracer has no CPU fallback")
        dev = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        if dev.index is None:
            dev = torch.device("cuda", torch.cuda.current_device())
        return dev

    def _bind(self, n_exp, ny, nx, device, stream):
        import torch
        self.torch = torch
        self.device = device
        self.shape = (n_exp, ny, nx) if n_exp > 1 or self._batch else (ny, nx)
        self.sum_p = torch.zeros(self.shape, dtype=torch.float64, device=self.device)
        self.sum_p2 = torch.zeros(self.shape, dtype=torch.float64, device=self.device)
        self.counts = torch.zeros(self.shape, dtype=torch.int64, device=self.device)  # bit pattern of uint64
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        _check(self.L, self.ctx, self.L.sas_bind_buffers(self.ctx, self.sum_p.data_ptr(), self.sum_p2.data_ptr(),
                                                         self.counts.data_ptr(), self.stream.cuda_stream))

    def reset(self):
        _check(self.L, self.ctx, self.L.sas_reset_detector(self.ctx))

    def counters(self):
        out = (C.c_uint64 * 8)()
        _check(self.L, self.ctx, self.L.sas_get_counters(self.ctx, out))
        return np.array(out[:], dtype=np.uint64)

    def read_detector(self):
        """Device -> host copy through the ABI: (sum_p, sum_p2, counts) numpy arrays (views of page-locked
        host buffers owned by this object and reused by the next call: copy what must outlive it)."""
        import torch
        if getattr(self, "_host", None) is None:   # page-locked once: the three copies are plain DMA transfers
            self._host = [torch.empty(self.shape, dtype=dt, pin_memory=True)
                          for dt in (torch.float64, torch.float64, torch.int64)]
        host = self._host
        _check(self.L, self.ctx, self.L.sas_read_detector(self.ctx, *(t.data_ptr() for t in host)))
        sp, sp2, cn = (t.numpy() for t in host)
        return sp, sp2, cn.view(np.uint64)

    def reduce_radial(self, lambda_ref, q_lo, q_hi, n_bins, exp_index=0, n_launched=0):
        """Ring average of the detector into I(q): (q, I, sigma, npix) numpy arrays (include/sas.h).
        n_launched: neutrons launched into that experiment held by the buffers (0 = this context's own count)."""
        d = RadialDesc(C.sizeof(RadialDesc), int(exp_index), int(n_bins), 0, float(q_lo), float(q_hi), float(lambda_ref),
                       int(n_launched))
        q, i, s = (np.zeros(max(n_bins, 1)) for _ in range(3))
        n = np.zeros(max(n_bins, 1), np.uint64)
        _check(self.L, self.ctx, self.L.sas_reduce_radial(self.ctx, C.byref(d), q.ctypes.data, i.ctypes.data,
                                                          s.ctypes.data, n.ctypes.data))
        return q, i, s, n

    def launch_info(self):
        n, g, b, s = C.c_uint64(), C.c_int32(), C.c_int32(), C.c_int32()
        _check(self.L, self.ctx, self.L.sas_get_launch_info(self.ctx, n, g, b, s))
        return dict(n_launches=n.value, grid=g.value, block=b.value, smem_bytes=s.value)

    def kernel_time_ms(self, reset=True):
        ms, n = C.c_double(), C.c_uint64()
        _check(self.L, self.ctx, self.L.sas_get_kernel_time(self.ctx, 1 if reset else 0, ms, n))
        return ms.value, n.value

    def set_launch_timing(self, enabled: bool):
        """Per-launch CUDA events on (default) or off (include/sas.h: sas_set_launch_timing)."""
        _check(self.L, self.ctx, self.L.sas_set_launch_timing(self.ctx, 1 if enabled else 0))

    def launch_records(self):
        """One dict per trace-kernel launch since the last kernel_time_ms(reset=True) (include/sas.h)."""
        buf = (LaunchRecord * MAX_LAUNCH_RECORDS)()
        n = C.c_uint32()
        _check(self.L, self.ctx, self.L.sas_get_launch_records(self.ctx, buf, MAX_LAUNCH_RECORDS, n))
        return [{k: getattr(buf[i], k) for k, _ in LaunchRecord._fields_} for i in range(min(n.value, MAX_LAUNCH_RECORDS))]

    def reduce_time_ms(self):
        ms = C.c_double()
        _check(self.L, self.ctx, self.L.sas_get_reduce_time(self.ctx, ms))
        return ms.value

    def upload_bytes(self):
        n = C.c_uint64()
        _check(self.L, self.ctx, self.L.sas_get_upload_bytes(self.ctx, n))
        return n.value

    def close(self):
        if getattr(self, "ctx", None):
            self.L.sas_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Tracer(_Base):
    """One virtual experiment: sas_create_instrument / sas_set_model / sas_trace / sas_read_detector."""
    _batch = False

    def __init__(self, instrument: dict, model: dict | None = None, device=None, stream=None):
        """device: a torch device (default: torch's current CUDA device, which is left unchanged)."""
        self.L = load_library()
        import torch
        dev = self._device(device)
        self.ctx = C.c_void_p()
        ins = instrument_desc(instrument)
        with torch.cuda.device(dev):       # the library creates the context on the calling thread's current device
            _check(self.L, None, self.L.sas_create_instrument(C.byref(ins), C.byref(self.ctx)))
        self._bind(1, ins.det_ny, ins.det_nx, dev, stream)
        if model is not None:
            self.set_model(model)

    def set_model(self, model: dict):
        m = model_desc(model)
        _check(self.L, self.ctx, self.L.sas_set_model(self.ctx, C.byref(m)))

    def trace(self, n_neutrons: int, seed: int):
        _check(self.L, self.ctx, self.L.sas_trace(self.ctx, n_neutrons, seed))

    def trace_range(self, first_id: int, n: int, seed: int):
        _check(self.L, self.ctx, self.L.sas_trace_range(self.ctx, first_id, n, seed))

    def trace_dump(self, first_id: int, n: int, seed: int, exp_index: int = 0, want_q: bool = True):
        """Parity hook: per-neutron (pixel, weight[, q]) as numpy arrays."""
        t = self.torch
        px = t.empty(n, dtype=t.int32, device=self.device)
        wt = t.empty(n, dtype=t.float64, device=self.device)
        qq = t.empty(n, dtype=t.float64, device=self.device) if want_q else None
        _check(self.L, self.ctx, self.L.sas_trace_dump(self.ctx, first_id, n, seed, exp_index, px.data_ptr(),
                                                       wt.data_ptr(), qq.data_ptr() if want_q else None))
        self.stream.synchronize()
        return px.cpu().numpy(), wt.cpu().numpy(), (qq.cpu().numpy() if want_q else None)


class BatchTracer(_Base):
    """Many experiments in one launch: sas_create_batch / sas_trace_batch."""
    _batch = True

    def __init__(self, instruments: list, models: list, device=None, stream=None):
        self.L = load_library()
        import torch
        dev = self._device(device)
        n = len(instruments)
        assert n == len(models) and n > 0
        ins = (InstrumentDesc * n)(*[instrument_desc(d) for d in instruments])
        mod = (ModelDesc * n)(*[model_desc(d) for d in models])
        self.ctx = C.c_void_p()
        with torch.cuda.device(dev):
            _check(self.L, None, self.L.sas_create_batch(ins, mod, n, C.byref(self.ctx)))
        self._bind(n, ins[0].det_ny, ins[0].det_nx, dev, stream)

    def trace(self, n_neutrons_each: int, seed: int):
        _check(self.L, self.ctx, self.L.sas_trace_batch(self.ctx, n_neutrons_each, seed))

    def trace_range(self, first_id: int, n_each: int, seed: int):
        """ids [first_id, first_id + n_each) of every experiment (resume, or one GPU's shard)."""
        _check(self.L, self.ctx, self.L.sas_trace_batch_range(self.ctx, first_id, n_each, seed))
