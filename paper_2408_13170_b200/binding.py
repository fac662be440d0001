"""ctypes binding of libscstat.so: the same names as include/sc_stat.h, argument marshalling only.

Device arguments are torch CUDA tensors (float64 / int32, contiguous); PyTorch is used for device memory and
streams, nothing else.  Calls go to the current torch CUDA stream unless `stream` is given.
If the library is missing or cannot be loaded every call raises SCError -- there is no fallback path.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libscstat.so")

SC_OK, SC_ERR_INVALID_ARG, SC_ERR_NOT_INIT, SC_ERR_CUDA, SC_ERR_OOM = 0, -1, -2, -3, -4
SC_OPT_PRECISION, SC_OPT_F32_MIN_SEG, SC_OPT_SCRATCH_BYTES, SC_OPT_TC_MAX_S, SC_OPT_STRIDE_LOG2, SC_OPT_PROFILE, SC_OPT_SINCOS, SC_OPT_MUFU_MIN_SEG = 1, 2, 3, 4, 5, 6, 7, 8
SC_OPT_ESCALATE, SC_OPT_ESC_TAU_POLY_X1000, SC_OPT_ESC_TAU_MUFU_X1000, SC_OPT_WINDOW_SORT = 9, 10, 11, 12
SC_OPT_TENSOR_CORES = 13
SC_OPT_FUSED_AET = 14
SC_OPT_WINDOW_FRACTION_PPM = 15
SC_OPT_QUAD_AMPLITUDES = 16
SC_TIMING_CLASSES = ["nodes", "dense", "stitch", "pso", "other", "escalation"]

EXPORTED_SYMBOLS = ["sc_init_data", "sc_init_data_host", "sc_init_data3", "sc_gen_template3", "sc_eval_stat", "sc_eval_stat_host", "sc_eval_segments",
                    "sc_eval_stat_adaptive", "sc_eval_components", "sc_eval_loglike", "sc_data_norm", "sc_gen_template", "sc_pso_step", "sc_pso_best", "sc_pso_pick", "sc_pso_move", "sc_pso_step_labeled", "sc_kmeans", "sc_kmeans_static", "sc_search_run", "sc_whiten_streams", "sc_eval_stat_streams", "sc_get_counters", "sc_get_launch_info", "sc_get_timing", "sc_measure_fp64_peak",
                    "sc_set_option", "sc_free",
                    "sc_last_error", "sc_version"]


class SCError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"scstat error {code}: {msg}")
        self.code = code


class ScConfig(C.Structure):
    """sc_config of include/sc_stat.h."""
    _fields_ = [("T_obs_s", C.c_double), ("j0", C.c_int64), ("n_bins", C.c_int64),
                ("n_channels", C.c_int32), ("window_mode", C.c_int32), ("pn_order_x2", C.c_int32),
                ("ecc_leading", C.c_int32), ("f_ref_ecc", C.c_double),
                ("arm_L_s", C.c_double), ("au_s", C.c_double), ("orbit_alpha0", C.c_double),
                ("orbit_lambda0", C.c_double), ("year_s", C.c_double)]

    @classmethod
    def from_dict(cls, d):
        c = cls()
        for k, _ in cls._fields_:
            setattr(c, k, d[k])
        return c


SC_MAX_RUNGS = 8


class ScSearchConfig(C.Structure):
    """sc_search_config of include/sc_stat.h."""
    _fields_ = [("n_rungs", C.c_int32), ("n_seg", C.c_int32 * SC_MAX_RUNGS),
                ("omega", C.c_double * SC_MAX_RUNGS), ("phi_p", C.c_double * SC_MAX_RUNGS), ("phi_g", C.c_double * SC_MAX_RUNGS),
                ("eps_min", (C.c_double * 8) * SC_MAX_RUNGS),
                ("adaptive_edges", C.c_int32), ("conv_window", C.c_int32), ("conv_delta", C.c_double),
                ("max_iters_per_rung", C.c_int32), ("kmeans_max_iters", C.c_int32), ("threshold", C.c_double),
                ("seed", C.c_uint64), ("ranking_precision", C.c_int32), ("reserved_", C.c_int32)]

    @classmethod
    def make(cls, ladder, hyper, adaptive_edges=True, conv_window=50, conv_delta=2.0, max_iters_per_rung=1000,
             kmeans_max_iters=100, threshold=100.0, seed=0, ranking_precision=0):
        """ladder: segment counts per rung; hyper: per rung a dict with omega, phi_p, phi_g, eps (8 values)."""
        c = cls()
        c.n_rungs = len(ladder)
        for r, (N, hp) in enumerate(zip(ladder, hyper)):
            c.n_seg[r] = int(N)
            c.omega[r], c.phi_p[r], c.phi_g[r] = float(hp["omega"]), float(hp["phi_p"]), float(hp["phi_g"])
            for m in range(8):
                c.eps_min[r][m] = float(hp["eps"][m])
        c.adaptive_edges, c.conv_window, c.conv_delta = int(bool(adaptive_edges)), int(conv_window), float(conv_delta)
        c.max_iters_per_rung, c.kmeans_max_iters = int(max_iters_per_rung), int(kmeans_max_iters)
        c.threshold, c.seed = float(threshold), int(seed) & (2 ** 64 - 1)
        c.ranking_precision, c.reserved_ = int(ranking_precision), 0
        return c


_lib = None
_vp = C.c_void_p


def library_path():
    return _LIB_PATH


def load_library():
    """Load libscstat.so (built by paper_2408_13170_b200.build / __graft_entry__.build()).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise SCError(SC_ERR_NOT_INIT, f"{_LIB_PATH} not built: run `python -m paper_2408_13170_b200.build` "
                                       "(needs nvcc); there is no CPU fallback")
    try:
        L = C.CDLL(_LIB_PATH)
    except OSError as e:
        raise SCError(SC_ERR_NOT_INIT, f"cannot load {_LIB_PATH}: {e}; there is no CPU fallback")
    cfgp = C.POINTER(ScConfig)
    L.sc_init_data.restype = C.c_int
    L.sc_init_data.argtypes = [C.POINTER(_vp), cfgp, _vp, _vp, _vp, _vp, _vp]
    L.sc_init_data3.restype = C.c_int
    L.sc_init_data3.argtypes = [C.POINTER(_vp), cfgp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]
    L.sc_gen_template3.restype = C.c_int
    L.sc_gen_template3.argtypes = [_vp, _vp, C.c_int64, _vp, _vp, _vp, _vp]
    L.sc_init_data_host.restype = C.c_int
    L.sc_init_data_host.argtypes = [C.POINTER(_vp), cfgp, _vp, _vp, _vp, _vp, _vp]
    for name in ("sc_eval_stat", "sc_eval_stat_host", "sc_eval_segments", "sc_eval_components"):
        f = getattr(L, name)
        f.restype = C.c_int
        f.argtypes = [_vp, _vp, C.c_int64, _vp, C.c_int32, _vp, _vp]
    L.sc_eval_stat_adaptive.restype = C.c_int
    L.sc_eval_stat_adaptive.argtypes = [_vp, _vp, C.c_int64, C.c_int32, _vp, _vp, _vp, _vp]
    L.sc_eval_loglike.restype = C.c_int
    L.sc_eval_loglike.argtypes = [_vp, _vp, _vp, C.c_int64, _vp, C.c_int32, _vp, _vp]
    L.sc_data_norm.restype = C.c_int
    L.sc_data_norm.argtypes = [_vp, C.POINTER(C.c_double)]
    L.sc_gen_template.restype = C.c_int
    L.sc_gen_template.argtypes = [_vp, _vp, C.c_int64, _vp, _vp, _vp]
    L.sc_pso_step.restype = C.c_int
    L.sc_pso_step.argtypes = [_vp] + [_vp] * 10 + [C.c_double] * 3 + [C.c_uint64, C.c_uint64, C.c_int64, C.c_int32, _vp]
    L.sc_pso_step_labeled.restype = C.c_int
    L.sc_pso_best.argtypes = [_vp] + [_vp] * 5 + [C.c_int64, C.c_int32, C.c_int64, _vp]
    L.sc_pso_pick.argtypes = [_vp, _vp, C.c_int32, C.c_int32, _vp, _vp, _vp]
    L.sc_pso_move.argtypes = [_vp] + [_vp] * 7 + [C.c_double] * 3 + [C.c_uint64, C.c_uint64, C.c_int64, C.c_int32, C.c_int64, _vp]
    L.sc_pso_step_labeled.argtypes = [_vp] + [_vp] * 11 + [C.c_double] * 3 + [C.c_uint64, C.c_uint64, C.c_int64, C.c_int32, _vp]
    L.sc_kmeans.restype = C.c_int
    L.sc_kmeans.argtypes = [_vp, _vp, C.c_int64, _vp, _vp, _vp, C.c_int32, C.c_int32, _vp, _vp, C.POINTER(C.c_int32), _vp]
    L.sc_kmeans_static.restype = C.c_int
    L.sc_kmeans_static.argtypes = L.sc_kmeans.argtypes
    L.sc_search_run.restype = C.c_int
    L.sc_search_run.argtypes = [_vp, C.POINTER(ScSearchConfig), _vp, _vp, _vp, C.c_int64, C.c_int32, _vp, _vp,
                                _vp, _vp, _vp, _vp, _vp, _vp, _vp]
    L.sc_whiten_streams.restype = C.c_int
    L.sc_whiten_streams.argtypes = [_vp, _vp, _vp, C.c_int64, C.c_int32, _vp, _vp]
    L.sc_eval_stat_streams.restype = C.c_int
    L.sc_eval_stat_streams.argtypes = [_vp, _vp, _vp, C.c_int32, C.c_int64, _vp, C.c_int32, _vp, _vp]
    L.sc_get_counters.restype = C.c_int
    L.sc_get_counters.argtypes = [_vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), _vp]
    L.sc_get_launch_info.restype = C.c_int
    L.sc_get_launch_info.argtypes = [_vp, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    L.sc_get_timing.restype = C.c_int
    L.sc_get_timing.argtypes = [_vp, C.POINTER(C.c_double), C.POINTER(C.c_int64), _vp]
    L.sc_measure_fp64_peak.restype = C.c_int
    L.sc_measure_fp64_peak.argtypes = [C.POINTER(C.c_double), _vp]
    L.sc_set_option.restype = C.c_int
    L.sc_set_option.argtypes = [_vp, C.c_int32, C.c_int64]
    L.sc_free.restype = C.c_int
    L.sc_free.argtypes = [_vp]
    L.sc_last_error.restype = C.c_char_p
    L.sc_last_error.argtypes = [_vp]
    L.sc_version.restype = C.c_char_p
    L.sc_version.argtypes = []
    _lib = L
    return L


def _torch():
    import torch
    return torch


def _stream(stream):
    if stream is not None:
        return _vp(int(stream))
    return _vp(int(_torch().cuda.current_stream().cuda_stream))


def _dev(t, dtype, name):
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise SCError(SC_ERR_INVALID_ARG, f"{name}: need a contiguous CUDA tensor of dtype {dtype}")
    return _vp(t.data_ptr())


def _host_f64(a, name):
    import numpy as np
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, _vp(a.ctypes.data)


def _edges_arg(seg_edges):
    """HOST numpy int32 array (preferred) or DEVICE int32 tensor -> (keepalive, pointer, n_seg)."""
    import numpy as np
    torch = _torch()
    if isinstance(seg_edges, torch.Tensor):
        if seg_edges.is_cuda:
            if seg_edges.dtype != torch.int32 or not seg_edges.is_contiguous():
                raise SCError(SC_ERR_INVALID_ARG, "seg_edges: device tensor must be contiguous int32")
            return seg_edges, _vp(seg_edges.data_ptr()), int(seg_edges.numel()) - 1
        seg_edges = seg_edges.numpy()
    e = np.ascontiguousarray(seg_edges)
    if e.size and (e.min() < -2 ** 31 or e.max() >= 2 ** 31):
        raise SCError(SC_ERR_INVALID_ARG, "seg_edges out of int32 range")
    e = e.astype(np.int32)
    return e, _vp(e.ctypes.data), int(e.size) - 1


def _check(rc, h):
    if rc != SC_OK:
        msg = load_library().sc_last_error(h)
        raise SCError(rc, msg.decode() if msg else "")


# ---------------------------------------------------------------------------------------------- C-named functions
def sc_version():
    return load_library().sc_version().decode()


def sc_last_error(h=None):
    m = load_library().sc_last_error(h)
    return m.decode() if m else ""


def sc_init_data(cfg, dA_ri, dE_ri, S_A, S_E, stream=None):
    """DEVICE float64 tensors: dA_ri, dE_ri [n_bins, 2] (re, im), S_A, S_E [n_bins].  Returns the opaque handle."""
    torch = _torch()
    L = load_library()
    if not isinstance(cfg, ScConfig):
        cfg = ScConfig.from_dict(cfg)
    n = int(cfg.n_bins)
    for t, m, nm in ((dA_ri, 2 * n, "dA_ri"), (dE_ri, 2 * n, "dE_ri"), (S_A, n, "S_A"), (S_E, n, "S_E")):
        if isinstance(t, torch.Tensor) and t.numel() != m:
            raise SCError(SC_ERR_INVALID_ARG, f"{nm}: expected {m} float64 values, got {t.numel()}")
    h = _vp()
    rc = L.sc_init_data(C.byref(h), C.byref(cfg), _dev(dA_ri, torch.float64, "dA_ri"), _dev(dE_ri, torch.float64, "dE_ri"),
                        _dev(S_A, torch.float64, "S_A"), _dev(S_E, torch.float64, "S_E"), _stream(stream))
    _check(rc, None)
    return h


def sc_init_data3(cfg, dA_ri, dE_ri, dT_ri, S_A, S_E, S_T, stream=None):
    """Three channels (A, E, T): DEVICE float64 tensors as in sc_init_data; cfg.n_channels must be 3."""
    torch = _torch()
    L = load_library()
    if not isinstance(cfg, ScConfig):
        cfg = ScConfig.from_dict(cfg)
    n = int(cfg.n_bins)
    names = ("dA_ri", "dE_ri", "dT_ri", "S_A", "S_E", "S_T")
    for t, m, nm in zip((dA_ri, dE_ri, dT_ri, S_A, S_E, S_T), (2 * n,) * 3 + (n,) * 3, names):
        if isinstance(t, torch.Tensor) and t.numel() != m:
            raise SCError(SC_ERR_INVALID_ARG, f"{nm}: expected {m} float64 values, got {t.numel()}")
    h = _vp()
    rc = L.sc_init_data3(C.byref(h), C.byref(cfg), *[_dev(t, torch.float64, nm) for t, nm in
                                                     zip((dA_ri, dE_ri, dT_ri, S_A, S_E, S_T), names)], _stream(stream))
    _check(rc, None)
    return h


def sc_gen_template3(h, params, n_templates, hA_ri, hE_ri, hT_ri, stream=None):
    torch = _torch()
    rc = load_library().sc_gen_template3(h, _dev(params, torch.float64, "params"), n_templates,
                                         _dev(hA_ri, torch.float64, "hA_ri"), _dev(hE_ri, torch.float64, "hE_ri"),
                                         _dev(hT_ri, torch.float64, "hT_ri"), _stream(stream))
    _check(rc, h)
    return hA_ri, hE_ri, hT_ri


def sc_init_data_host(cfg, dA, dE, S_A, S_E, stream=None):
    """HOST numpy arrays: dA, dE complex128 [n_bins] (or float64 [n_bins, 2]); S_A, S_E float64 [n_bins]."""
    import numpy as np
    L = load_library()
    if not isinstance(cfg, ScConfig):
        cfg = ScConfig.from_dict(cfg)
    n = int(cfg.n_bins)
    arrs = []
    for a, m, nm in ((dA, 2 * n, "dA"), (dE, 2 * n, "dE"), (S_A, n, "S_A"), (S_E, n, "S_E")):
        a = np.ascontiguousarray(a)
        if np.iscomplexobj(a):
            a = np.ascontiguousarray(a, dtype=np.complex128).view(np.float64)
        a = np.ascontiguousarray(a, dtype=np.float64)
        if a.size != m:
            raise SCError(SC_ERR_INVALID_ARG, f"{nm}: expected {m} float64 values, got {a.size}")
        arrs.append(a)
    h = _vp()
    rc = L.sc_init_data_host(C.byref(h), C.byref(cfg), *[_vp(a.ctypes.data) for a in arrs], _stream(stream))
    _check(rc, None)
    return h


def sc_eval_stat(h, params, n_particles, seg_edges, n_seg, out, stream=None):
    torch = _torch()
    keep, ep, ns = _edges_arg(seg_edges)
    if ns != n_seg:
        raise SCError(SC_ERR_INVALID_ARG, f"seg_edges has {ns + 1} entries, expected n_seg + 1 = {n_seg + 1}")
    if params.numel() != 8 * n_particles or out.numel() != n_particles:
        raise SCError(SC_ERR_INVALID_ARG, "params must be [n_particles, 8] and out [n_particles]")
    rc = load_library().sc_eval_stat(h, _dev(params, torch.float64, "params"), n_particles, ep, n_seg,
                                     _dev(out, torch.float64, "out"), _stream(stream))
    _check(rc, h)
    return out


def sc_eval_stat_host(h, params, n_particles, seg_edges, n_seg, out, stream=None):
    """HOST numpy params [n_particles, 8] / out [n_particles] (float64); copies run inside the C call."""
    import numpy as np
    keep, ep, ns = _edges_arg(seg_edges)
    if ns != n_seg:
        raise SCError(SC_ERR_INVALID_ARG, f"seg_edges has {ns + 1} entries, expected n_seg + 1 = {n_seg + 1}")
    if not (isinstance(params, np.ndarray) and params.dtype == np.float64 and params.flags.c_contiguous
            and params.size == 8 * n_particles):
        raise SCError(SC_ERR_INVALID_ARG, "params: need C-contiguous float64 numpy [n_particles, 8]")
    if not (isinstance(out, np.ndarray) and out.dtype == np.float64 and out.flags.c_contiguous and out.size == n_particles):
        raise SCError(SC_ERR_INVALID_ARG, "out: need C-contiguous float64 numpy [n_particles]")
    rc = load_library().sc_eval_stat_host(h, _vp(params.ctypes.data), n_particles, ep, n_seg, _vp(out.ctypes.data),
                                          _stream(stream))
    _check(rc, h)
    return out


def sc_eval_segments(h, params, n_particles, seg_edges, n_seg, out_seg, stream=None):
    torch = _torch()
    keep, ep, ns = _edges_arg(seg_edges)
    if ns != n_seg:
        raise SCError(SC_ERR_INVALID_ARG, f"seg_edges has {ns + 1} entries, expected n_seg + 1 = {n_seg + 1}")
    if params.numel() != 8 * n_particles or out_seg.numel() != n_particles * n_seg * 3:
        raise SCError(SC_ERR_INVALID_ARG, "params must be [n_particles, 8] and out_seg [n_particles, n_seg, 3]")
    rc = load_library().sc_eval_segments(h, _dev(params, torch.float64, "params"), n_particles, ep, n_seg,
                                         _dev(out_seg, torch.float64, "out_seg"), _stream(stream))
    _check(rc, h)
    return out_seg


def sc_eval_stat_adaptive(h, params, n_particles, n_seg, out=None, out_edges=None, out3=None, stream=None):
    """Per-particle equal-SNR^2 segments.  out [P] f64, out_edges [P, n_seg+1] int32, out3 [P, 3] f64:
    CUDA tensors or None (at least one of out / out3)."""
    torch = _torch()
    if params.numel() != 8 * n_particles:
        raise SCError(SC_ERR_INVALID_ARG, "params must be [n_particles, 8]")
    for t, sz, nm in ((out, n_particles, "out"), (out_edges, n_particles * (n_seg + 1), "out_edges"), (out3, 3 * n_particles, "out3")):
        if t is not None and t.numel() != sz:
            raise SCError(SC_ERR_INVALID_ARG, f"{nm}: expected {sz} values, got {t.numel()}")
    rc = load_library().sc_eval_stat_adaptive(
        h, _dev(params, torch.float64, "params"), n_particles, n_seg,
        None if out is None else _dev(out, torch.float64, "out"),
        None if out_edges is None else _dev(out_edges, torch.int32, "out_edges"),
        None if out3 is None else _dev(out3, torch.float64, "out3"), _stream(stream))
    _check(rc, h)
    return out, out_edges, out3


def sc_eval_components(h, params, n_particles, seg_edges, n_seg, out3, stream=None):
    torch = _torch()
    keep, ep, ns = _edges_arg(seg_edges)
    if ns != n_seg:
        raise SCError(SC_ERR_INVALID_ARG, f"seg_edges has {ns + 1} entries, expected n_seg + 1 = {n_seg + 1}")
    if params.numel() != 8 * n_particles or out3.numel() != n_particles * 3:
        raise SCError(SC_ERR_INVALID_ARG, "params must be [n_particles, 8] and out3 [n_particles, 3]")
    rc = load_library().sc_eval_components(h, _dev(params, torch.float64, "params"), n_particles, ep, n_seg,
                                           _dev(out3, torch.float64, "out3"), _stream(stream))
    _check(rc, h)
    return out3


def sc_eval_loglike(h, params, amp, n_particles, seg_edges, n_seg, out, stream=None):
    torch = _torch()
    keep, ep, ns = _edges_arg(seg_edges)
    if ns != n_seg:
        raise SCError(SC_ERR_INVALID_ARG, f"seg_edges has {ns + 1} entries, expected n_seg + 1 = {n_seg + 1}")
    if params.numel() != 8 * n_particles or amp.numel() != n_particles or out.numel() != n_particles:
        raise SCError(SC_ERR_INVALID_ARG, "params must be [n_particles, 8], amp and out [n_particles]")
    rc = load_library().sc_eval_loglike(h, _dev(params, torch.float64, "params"), _dev(amp, torch.float64, "amp"),
                                        n_particles, ep, n_seg, _dev(out, torch.float64, "out"), _stream(stream))
    _check(rc, h)
    return out


def sc_data_norm(h):
    v = C.c_double(0.0)
    _check(load_library().sc_data_norm(h, C.byref(v)), h)
    return v.value


def sc_gen_template(h, params, n_templates, hA_ri, hE_ri, stream=None):
    torch = _torch()
    rc = load_library().sc_gen_template(h, _dev(params, torch.float64, "params"), n_templates,
                                        _dev(hA_ri, torch.float64, "hA_ri"), _dev(hE_ri, torch.float64, "hE_ri"),
                                        _stream(stream))
    _check(rc, h)
    return hA_ri, hE_ri


def sc_pso_step(h, pos, vel, pbest_pos, pbest_val, stat, gbest_pos, gbest_val, lo, hi, eps_min,
                omega, phi_p, phi_g, seed, iter, n_particles, n_swarms, stream=None):
    torch = _torch()
    names = ["pos", "vel", "pbest_pos", "pbest_val", "stat", "gbest_pos", "gbest_val", "lo", "hi", "eps_min"]
    tens = [pos, vel, pbest_pos, pbest_val, stat, gbest_pos, gbest_val, lo, hi, eps_min]
    sizes = [8 * n_particles] * 3 + [n_particles] * 2 + [8 * n_swarms, n_swarms, 8, 8, 8]
    for t, nm, sz in zip(tens, names, sizes):
        if isinstance(t, torch.Tensor) and t.numel() != sz:
            raise SCError(SC_ERR_INVALID_ARG, f"{nm}: expected {sz} values, got {t.numel()}")
    ptrs = [_dev(t, torch.float64, nm) for t, nm in zip(tens, names)]
    rc = load_library().sc_pso_step(h, *ptrs, float(omega), float(phi_p), float(phi_g), int(seed) & (2 ** 64 - 1),
                                    int(iter), int(n_particles), int(n_swarms), _stream(stream))
    _check(rc, h)


def sc_pso_best(h, pos, pbest_pos, pbest_val, stat, cand, n_particles, n_swarms, index_offset=0, stream=None):
    torch = _torch()
    names = ["pos", "pbest_pos", "pbest_val", "stat", "cand"]
    tens = [pos, pbest_pos, pbest_val, stat, cand]
    sizes = [8 * n_particles] * 2 + [n_particles] * 2 + [10 * n_swarms]
    for t, nm, sz in zip(tens, names, sizes):
        if t.numel() != sz:
            raise SCError(SC_ERR_INVALID_ARG, f"{nm}: expected {sz} values, got {t.numel()}")
    ptrs = [_dev(t, torch.float64, nm) for t, nm in zip(tens, names)]
    _check(load_library().sc_pso_best(h, *ptrs, int(n_particles), int(n_swarms), int(index_offset), _stream(stream)), h)


def sc_pso_pick(h, cand, n_cand, n_swarms, gbest_pos, gbest_val, stream=None):
    torch = _torch()
    if cand.numel() != 10 * n_cand * n_swarms or gbest_pos.numel() != 8 * n_swarms or gbest_val.numel() != n_swarms:
        raise SCError(SC_ERR_INVALID_ARG, "cand [n_cand, n_swarms, 10], gbest_pos [n_swarms, 8], gbest_val [n_swarms] expected")
    _check(load_library().sc_pso_pick(h, _dev(cand, torch.float64, "cand"), int(n_cand), int(n_swarms),
                                      _dev(gbest_pos, torch.float64, "gbest_pos"), _dev(gbest_val, torch.float64, "gbest_val"),
                                      _stream(stream)), h)


def sc_pso_move(h, pos, vel, pbest_pos, gbest_pos, lo, hi, eps_min, omega, phi_p, phi_g, seed, iter, n_particles, n_swarms,
                index_offset=0, stream=None):
    torch = _torch()
    names = ["pos", "vel", "pbest_pos", "gbest_pos", "lo", "hi", "eps_min"]
    tens = [pos, vel, pbest_pos, gbest_pos, lo, hi, eps_min]
    sizes = [8 * n_particles] * 3 + [8 * n_swarms, 8, 8, 8]
    for t, nm, sz in zip(tens, names, sizes):
        if t.numel() != sz:
            raise SCError(SC_ERR_INVALID_ARG, f"{nm}: expected {sz} values, got {t.numel()}")
    ptrs = [_dev(t, torch.float64, nm) for t, nm in zip(tens, names)]
    _check(load_library().sc_pso_move(h, *ptrs, float(omega), float(phi_p), float(phi_g), int(seed) & (2 ** 64 - 1), int(iter),
                                      int(n_particles), int(n_swarms), int(index_offset), _stream(stream)), h)


def sc_pso_step_labeled(h, pos, vel, pbest_pos, pbest_val, stat, gbest_pos, gbest_val, label, lo, hi, eps_min,
                        omega, phi_p, phi_g, seed, iter, n_particles, n_swarms, stream=None):
    torch = _torch()
    names = ["pos", "vel", "pbest_pos", "pbest_val", "stat", "gbest_pos", "gbest_val", "lo", "hi", "eps_min"]
    tens = [pos, vel, pbest_pos, pbest_val, stat, gbest_pos, gbest_val, lo, hi, eps_min]
    sizes = [8 * n_particles] * 3 + [n_particles] * 2 + [8 * n_swarms, n_swarms, 8, 8, 8]
    for t, nm, sz in zip(tens, names, sizes):
        if isinstance(t, torch.Tensor) and t.numel() != sz:
            raise SCError(SC_ERR_INVALID_ARG, f"{nm}: expected {sz} values, got {t.numel()}")
    if label.numel() != n_particles:
        raise SCError(SC_ERR_INVALID_ARG, "label: expected n_particles int32 values")
    ptrs = [_dev(t, torch.float64, nm) for t, nm in zip(tens, names)]
    ptrs.insert(7, _dev(label, torch.int32, "label"))
    rc = load_library().sc_pso_step_labeled(h, *ptrs, float(omega), float(phi_p), float(phi_g), int(seed) & (2 ** 64 - 1),
                                            int(iter), int(n_particles), int(n_swarms), _stream(stream))
    _check(rc, h)


def sc_kmeans(h, pos, n_particles, lo, hi, cent, K, max_iter, label, count=None, stream=None):
    """-> iterations run.  All tensors CUDA: pos [P,8], lo/hi [8], cent [K,8] (in/out) f64; label [P] int32; count [K] int64."""
    torch = _torch()
    if pos.numel() != 8 * n_particles or cent.numel() != 8 * K or label.numel() != n_particles:
        raise SCError(SC_ERR_INVALID_ARG, "pos [P,8], cent [K,8], label [P] expected")
    n_it = C.c_int32(0)
    rc = load_library().sc_kmeans(h, _dev(pos, torch.float64, "pos"), n_particles, _dev(lo, torch.float64, "lo"),
                                  _dev(hi, torch.float64, "hi"), _dev(cent, torch.float64, "cent"), K, max_iter,
                                  _dev(label, torch.int32, "label"),
                                  None if count is None else _dev(count, torch.int64, "count"), C.byref(n_it), _stream(stream))
    _check(rc, h)
    return n_it.value


SC_KMEANS_STATIC_MAX_K = 128


def sc_kmeans_static(h, pos, n_particles, lo, hi, cent, K, max_iter, label, count=None, stream=None):
    """sc_kmeans without device allocation (scratch in a static device array of the library, K <= SC_KMEANS_STATIC_MAX_K);
    same arguments and results.  Calls that overlap on the GPU race: the array is shared."""
    torch = _torch()
    if pos.numel() != 8 * n_particles or cent.numel() != 8 * K or label.numel() != n_particles:
        raise SCError(SC_ERR_INVALID_ARG, "pos [P,8], cent [K,8], label [P] expected")
    n_it = C.c_int32(0)
    rc = load_library().sc_kmeans_static(h, _dev(pos, torch.float64, "pos"), n_particles, _dev(lo, torch.float64, "lo"),
                                         _dev(hi, torch.float64, "hi"), _dev(cent, torch.float64, "cent"), K, max_iter,
                                         _dev(label, torch.int32, "label"),
                                         None if count is None else _dev(count, torch.int64, "count"), C.byref(n_it), _stream(stream))
    _check(rc, h)
    return n_it.value


def sc_search_run(h, cfg, pos, vel, label, n_particles, n_swarms, lo, hi, stream=None):
    """Runs the ladder on the device; pos, vel, label are updated in place.  Returns a dict of HOST numpy results."""
    import numpy as np
    torch = _torch()
    if pos.numel() != 8 * n_particles or vel.numel() != 8 * n_particles or label.numel() != n_particles:
        raise SCError(SC_ERR_INVALID_ARG, "pos, vel [P,8] and label [P] expected")
    S, R, M = int(n_swarms), int(cfg.n_rungs), int(cfg.max_iters_per_rung)
    best_pos, best_val = np.zeros((S, 8)), np.zeros(S)
    n_members, passed = np.zeros(S, dtype=np.int64), np.zeros(S, dtype=np.int32)
    iters, hist = np.zeros(max(R, 1), dtype=np.int32), np.zeros((max(R, 1), S, max(M, 1)))
    p = lambda a: _vp(a.ctypes.data)
    rc = load_library().sc_search_run(h, C.byref(cfg), _dev(pos, torch.float64, "pos"), _dev(vel, torch.float64, "vel"),
                                      _dev(label, torch.int32, "label"), n_particles, S, _dev(lo, torch.float64, "lo"),
                                      _dev(hi, torch.float64, "hi"), p(best_pos), p(best_val), p(n_members), p(passed),
                                      p(iters), p(hist), _stream(stream))
    _check(rc, h)
    return dict(best_pos=best_pos, best_val=best_val, n_members=n_members, passed=passed, iters_per_rung=iters, hist=hist)


def sc_whiten_streams(h, dA_ri, dE_ri, n_streams, W, stream=None):
    """dA_ri, dE_ri: CUDA f64 [n_streams, n_bins, 2]; W: CUDA [n_streams, n_bins, 4] float32 or float64 (out)."""
    torch = _torch()
    if W.dtype not in (torch.float32, torch.float64):
        raise SCError(SC_ERR_INVALID_ARG, "W must be float32 or float64")
    if dA_ri.numel() != dE_ri.numel() or W.numel() != 2 * dA_ri.numel() or dA_ri.numel() % (2 * n_streams):
        raise SCError(SC_ERR_INVALID_ARG, "expected dA_ri, dE_ri [n_streams, n_bins, 2] and W [n_streams, n_bins, 4]")
    rc = load_library().sc_whiten_streams(h, _dev(dA_ri, torch.float64, "dA_ri"), _dev(dE_ri, torch.float64, "dE_ri"),
                                          n_streams, int(W.dtype == torch.float64), _dev(W, W.dtype, "W"), _stream(stream))
    _check(rc, h)
    return W


def sc_eval_stat_streams(h, theta, W, n_streams, seg_edges, n_seg, out, stream=None):
    torch = _torch()
    keep, ep, ns = _edges_arg(seg_edges)
    if ns != n_seg:
        raise SCError(SC_ERR_INVALID_ARG, f"seg_edges has {ns + 1} entries, expected n_seg + 1 = {n_seg + 1}")
    if theta.numel() != 8 or out.numel() != n_streams or W.dtype not in (torch.float32, torch.float64) or W.numel() % (4 * n_streams):
        raise SCError(SC_ERR_INVALID_ARG, "theta [8], W [n_streams, n_bins, 4] (float32/float64), out [n_streams] expected")
    rc = load_library().sc_eval_stat_streams(h, _dev(theta, torch.float64, "theta"), _dev(W, W.dtype, "W"),
                                             int(W.dtype == torch.float64), n_streams, ep, n_seg,
                                             _dev(out, torch.float64, "out"), _stream(stream))
    _check(rc, h)
    return out


def sc_get_counters(h, stream=None):
    """(evaluated_bins of the last eval, kernel launches since init); synchronises the stream."""
    a, b = C.c_int64(0), C.c_int64(0)
    rc = load_library().sc_get_counters(h, C.byref(a), C.byref(b), _stream(stream))
    _check(rc, h)
    return a.value, b.value


SC_FLAVOUR_MUFU, SC_FLAVOUR_MERGE, SC_FLAVOUR_QUAD, SC_FLAVOUR_TC, SC_FLAVOUR_AET = 1, 2, 4, 8, 16


def sc_get_launch_info(h):
    """(log2 node spacing, flavour bits) of the last FP32-amplitude pass."""
    a, b = C.c_int32(0), C.c_int32(0)
    _check(load_library().sc_get_launch_info(h, C.byref(a), C.byref(b)), h)
    return a.value, b.value


def sc_get_timing(h, stream=None):
    """{class: (ms, launches)} since the previous call (needs SC_OPT_PROFILE = 1); synchronises the stream."""
    ms = (C.c_double * len(SC_TIMING_CLASSES))()
    n = (C.c_int64 * len(SC_TIMING_CLASSES))()
    _check(load_library().sc_get_timing(h, ms, n, _stream(stream)), h)
    return {k: (ms[i], n[i]) for i, k in enumerate(SC_TIMING_CLASSES)}


def sc_measure_fp64_peak(stream=None):
    v = C.c_double(0.0)
    _check(load_library().sc_measure_fp64_peak(C.byref(v), _stream(stream)), None)
    return v.value


def sc_set_option(h, option, value):
    _check(load_library().sc_set_option(h, int(option), int(value)), h)


def sc_free(h):
    if h is not None and h.value:
        load_library().sc_free(h)
        h.value = None


# ---------------------------------------------------------------------------------------------- convenience wrapper
class Handle:
    """Owns one sc_handle.  Methods forward to the C-named functions above."""

    def __init__(self, cfg, dA, dE, S_A, S_E, host=False, stream=None, dT=None, S_T=None):
        self.cfg = cfg if isinstance(cfg, ScConfig) else ScConfig.from_dict(cfg)
        if dT is not None:                      # three channels (A, E, T)
            self.h = sc_init_data3(self.cfg, dA, dE, dT, S_A, S_E, S_T, stream)
        else:
            self.h = (sc_init_data_host if host else sc_init_data)(self.cfg, dA, dE, S_A, S_E, stream)

    def eval_stat(self, params, seg_edges, out=None, stream=None):
        torch = _torch()
        P = params.shape[0]
        if out is None:
            out = torch.empty(P, dtype=torch.float64, device=params.device)
        return sc_eval_stat(self.h, params, P, seg_edges, len(seg_edges) - 1, out, stream)

    def eval_stat_host(self, params, seg_edges, out=None, stream=None):
        import numpy as np
        P = params.shape[0]
        if out is None:
            out = np.empty(P, dtype=np.float64)
        return sc_eval_stat_host(self.h, params, P, seg_edges, len(seg_edges) - 1, out, stream)

    def eval_segments(self, params, seg_edges, stream=None):
        torch = _torch()
        P, N = params.shape[0], len(seg_edges) - 1
        out = torch.empty((P, N, 3), dtype=torch.float64, device=params.device)
        return sc_eval_segments(self.h, params, P, seg_edges, N, out, stream)

    def eval_stat_adaptive(self, params, n_seg, want_edges=False, want_comp=False, stream=None):
        """Upsilon_N on per-particle equal-SNR^2 segments -> out [P] (, edges [P, n_seg+1] int32) (, comp [P, 3])."""
        torch = _torch()
        P = params.shape[0]
        out = torch.empty(P, dtype=torch.float64, device=params.device)
        ed = torch.empty((P, n_seg + 1), dtype=torch.int32, device=params.device) if want_edges else None
        c3 = torch.empty((P, 3), dtype=torch.float64, device=params.device) if want_comp else None
        sc_eval_stat_adaptive(self.h, params, P, n_seg, out, ed, c3, stream)
        res = [out] + ([ed] if want_edges else []) + ([c3] if want_comp else [])
        return res[0] if len(res) == 1 else tuple(res)

    def eval_components(self, params, seg_edges, stream=None):
        """-> CUDA tensor [P, 3] = (Upsilon_N, O_hat_N, <h|h>)  (Eq. 10, 8, 3)."""
        torch = _torch()
        P = params.shape[0]
        out = torch.empty((P, 3), dtype=torch.float64, device=params.device)
        return sc_eval_components(self.h, params, P, seg_edges, len(seg_edges) - 1, out, stream)

    def eval_loglike(self, params, amp, seg_edges, stream=None):
        """-> CUDA tensor [P] = log L_hat_N (Eq. 9) for template amplitudes amp [P]."""
        torch = _torch()
        P = params.shape[0]
        out = torch.empty(P, dtype=torch.float64, device=params.device)
        return sc_eval_loglike(self.h, params, amp, P, seg_edges, len(seg_edges) - 1, out, stream)

    def data_norm(self):
        return sc_data_norm(self.h)

    def gen_template(self, params, stream=None):
        """-> (h_A, h_E) complex128 CUDA tensors [n_templates, n_bins]."""
        torch = _torch()
        params = params.reshape(-1, 8)
        n = int(self.cfg.n_bins)
        hA = torch.empty((params.shape[0], n, 2), dtype=torch.float64, device=params.device)
        hE = torch.empty_like(hA)
        sc_gen_template(self.h, params, params.shape[0], hA, hE, stream)
        return torch.view_as_complex(hA), torch.view_as_complex(hE)

    def gen_template3(self, params, stream=None):
        """-> (h_A, h_E, h_T) complex128 CUDA tensors [n_templates, n_bins] (three-channel handles)."""
        torch = _torch()
        params = params.reshape(-1, 8)
        n = int(self.cfg.n_bins)
        h3 = [torch.empty((params.shape[0], n, 2), dtype=torch.float64, device=params.device) for _ in range(3)]
        sc_gen_template3(self.h, params, params.shape[0], *h3, stream)
        return tuple(torch.view_as_complex(x) for x in h3)

    def pso_step(self, state, stat, lo, hi, eps_min, omega, phi_p, phi_g, seed, it, n_swarms, stream=None):
        """state: dict of CUDA tensors pos, vel, pbest_pos, pbest_val, gbest_pos, gbest_val (updated in place)."""
        sc_pso_step(self.h, state["pos"], state["vel"], state["pbest_pos"], state["pbest_val"], stat,
                    state["gbest_pos"], state["gbest_val"], lo, hi, eps_min, omega, phi_p, phi_g, seed, it,
                    state["pos"].shape[0], n_swarms, stream)

    def pso_best(self, state, stat, cand, n_swarms, index_offset=0, stream=None):
        """Steps (1)-(2) of sc_pso_step on this rank's particles -> cand [n_swarms, 10] (see sc_pso_best)."""
        sc_pso_best(self.h, state["pos"], state["pbest_pos"], state["pbest_val"], stat, cand, state["pos"].shape[0], n_swarms,
                    index_offset, stream)

    def pso_pick(self, cand, state, stream=None):
        """cand [n_cand, n_swarms, 10] -> state["gbest_pos"], state["gbest_val"]."""
        sc_pso_pick(self.h, cand, cand.shape[0], state["gbest_val"].shape[0], state["gbest_pos"], state["gbest_val"], stream)

    def pso_move(self, state, lo, hi, eps_min, omega, phi_p, phi_g, seed, it, n_swarms, index_offset=0, stream=None):
        sc_pso_move(self.h, state["pos"], state["vel"], state["pbest_pos"], state["gbest_pos"], lo, hi, eps_min, omega, phi_p,
                    phi_g, seed, it, state["pos"].shape[0], n_swarms, index_offset, stream)

    def pso_step_labeled(self, state, stat, label, lo, hi, eps_min, omega, phi_p, phi_g, seed, it, stream=None):
        sc_pso_step_labeled(self.h, state["pos"], state["vel"], state["pbest_pos"], state["pbest_val"], stat,
                            state["gbest_pos"], state["gbest_val"], label, lo, hi, eps_min, omega, phi_p, phi_g, seed, it,
                            state["pos"].shape[0], state["gbest_val"].shape[0], stream)

    def kmeans(self, pos, lo, hi, cent, max_iter=100, stream=None):
        """-> (label int32 [P], count int64 [K], iterations); cent [K,8] is updated in place."""
        torch = _torch()
        P, K = pos.shape[0], cent.shape[0]
        label = torch.empty(P, dtype=torch.int32, device=pos.device)
        count = torch.empty(K, dtype=torch.int64, device=pos.device)
        it = sc_kmeans(self.h, pos, P, lo, hi, cent, K, max_iter, label, count, stream)
        return label, count, it

    def search_run(self, cfg, pos, vel, label, n_swarms, lo, hi, stream=None):
        return sc_search_run(self.h, cfg, pos, vel, label, pos.shape[0], n_swarms, lo, hi, stream)

    def whiten_streams(self, dA, dE, f64=False, stream=None):
        """dA, dE: CUDA complex128 [n_streams, n_bins] -> whitened W [n_streams, n_bins, 4] (float32 or float64)."""
        torch = _torch()
        D, n = dA.shape
        W = torch.empty((D, n, 4), dtype=torch.float64 if f64 else torch.float32, device=dA.device)
        return sc_whiten_streams(self.h, torch.view_as_real(dA).contiguous(), torch.view_as_real(dE).contiguous(), D, W, stream)

    def eval_stat_streams(self, theta, W, seg_edges, out=None, stream=None):
        """Upsilon_N of ONE template (theta [8]) against every stream of W -> [n_streams]."""
        torch = _torch()
        D = W.shape[0]
        if out is None:
            out = torch.empty(D, dtype=torch.float64, device=W.device)
        return sc_eval_stat_streams(self.h, theta, W, D, seg_edges, len(seg_edges) - 1, out, stream)

    def counters(self, stream=None):
        return sc_get_counters(self.h, stream)

    def timing(self, stream=None):
        return sc_get_timing(self.h, stream)

    def launch_info(self):
        return sc_get_launch_info(self.h)

    def set_option(self, option, value):
        sc_set_option(self.h, option, value)

    def close(self):
        sc_free(self.h)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
