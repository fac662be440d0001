"""ctypes binding of the CPU ORACLE (oracle/sc_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It shares no code with paper_2408_13170_b200/ and neither imports the other.
Argument marshalling only: every number is computed by the C file beside it.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sc_oracle.c")
_LIB = os.path.join(_HERE, "libsc_oracle.so")


def build(force=False):
    """Compile the oracle with gcc (plain FP64, no contraction, OpenMP over particles)."""
    deps = [_SRC, os.path.join(_HERE, "sc_oracle.h")]
    if (not force and os.path.exists(_LIB)
            and all(os.path.getmtime(_LIB) >= os.path.getmtime(d) for d in deps)):
        return _LIB
    subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall",
                           "-o", _LIB, _SRC, "-lm"])
    return _LIB


class Config(C.Structure):
    _fields_ = [("T_obs_s", C.c_double), ("j0", C.c_int64), ("n_bins", C.c_int64),
                ("n_channels", C.c_int32), ("window_mode", C.c_int32), ("pn_order_x2", C.c_int32),
                ("ecc_leading", C.c_int32), ("f_ref_ecc", C.c_double),
                ("arm_L_s", C.c_double), ("au_s", C.c_double), ("orbit_alpha0", C.c_double),
                ("orbit_lambda0", C.c_double), ("year_s", C.c_double),
                ("truth_mode", C.c_int32), ("reserved_", C.c_int32)]


def make_config(d, truth=False):
    """d: dict with the field names above (what sc_synth.grid_config returns).  truth=True: long-double phase mode."""
    c = Config()
    for k, _ in Config._fields_:
        setattr(c, k, d.get(k, 0))
    c.truth_mode = 1 if truth else 0
    return c


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int64)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        L.sco_phase.restype = C.c_double
        L.sco_phase.argtypes = [C.POINTER(Config), _dp, C.c_double]
        L.sco_tf.restype = C.c_double
        L.sco_tf.argtypes = [C.POINTER(Config), _dp, C.c_double]
        L.sco_phase_truth.argtypes = [C.POINTER(Config), _dp, C.c_int64, _dp]
        L.sco_tf_truth.restype = C.c_double
        L.sco_tf_truth.argtypes = [C.POINTER(Config), _dp, C.c_int64]
        L.sco_orbit.argtypes = [C.POINTER(Config), C.c_double, _dp]
        L.sco_link.argtypes = [C.POINTER(Config), _dp, C.c_double, C.c_double, C.c_int, C.c_int, _dp]
        L.sco_tdi.argtypes = [C.POINTER(Config), _dp, C.c_double, C.c_double, _dp]
        L.sco_template.restype = C.c_int64
        L.sco_template.argtypes = [C.POINTER(Config), _dp, C.c_int64, C.c_int64, _dp, _dp]
        L.sco_stat_from_arrays.restype = C.c_double
        L.sco_stat_from_arrays.argtypes = [_dp, _dp, _dp, _dp, _dp, _dp, C.c_double, _ip, C.c_int64, _dp]
        L.sco_inner.restype = C.c_double
        L.sco_inner.argtypes = [_dp, _dp, _dp, _dp, _dp, _dp, C.c_double, C.c_int64]
        L.sco_eval_stat.argtypes = [C.POINTER(Config), _dp, _dp, _dp, _dp, _dp, C.c_int64, _ip, C.c_int64,
                                    _dp, _dp, _ip]
        L.sco_eval_stat_levels.argtypes = [C.POINTER(Config), _dp, _dp, _dp, _dp, _dp, C.c_int64, _ip, _ip,
                                           C.c_int64, _dp]
        L.sco_components_from_seg.argtypes = [_dp, C.c_int64, C.c_double, _dp]
        L.sco_loglike.restype = C.c_double
        L.sco_loglike.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double]
        L.sco_equal_snr_edges.argtypes = [_dp, _dp, _dp, _dp, C.c_int64, C.c_int64, _ip]
        L.sco_eval_stat_adaptive.argtypes = [C.POINTER(Config), _dp, _dp, _dp, _dp, _dp, C.c_int64, C.c_int64, _ip,
                                             _dp, _ip, _dp]
        L.sco_num_threads.restype = C.c_int
        L.sco_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.sco_pso_uniforms.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, _dp, _dp]
        L.sco_pso_step.argtypes = [_dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp,
                                   C.c_double, C.c_double, C.c_double, C.c_uint64, C.c_uint64, C.c_int64, C.c_int32]
        _i32p = C.POINTER(C.c_int32)
        L.sco_pso_step_labeled.argtypes = [_dp, _dp, _dp, _dp, _dp, _dp, _dp, _i32p, _dp, _dp, _dp,
                                           C.c_double, C.c_double, C.c_double, C.c_uint64, C.c_uint64, C.c_int64, C.c_int32]
        L.sco_kmeans.restype = C.c_int32
        L.sco_kmeans.argtypes = [_dp, C.c_int64, _dp, _dp, _dp, C.c_int32, C.c_int32, _i32p, _ip]
        L.sco_template3.restype = C.c_int64
        L.sco_template3.argtypes = [C.POINTER(Config), _dp, C.c_int64, C.c_int64, _dp, _dp, _dp]
        L.sco_stat_from_arrays3.restype = C.c_double
        L.sco_stat_from_arrays3.argtypes = [_dp] * 9 + [C.c_double, _ip, C.c_int64, _dp]
        L.sco_inner3.restype = C.c_double
        L.sco_inner3.argtypes = [_dp] * 9 + [C.c_double, C.c_int64]
        L.sco_eval_stat3.argtypes = [C.POINTER(Config)] + [_dp] * 7 + [C.c_int64, _ip, C.c_int64, _dp, _dp]
        L.sco_equal_snr_edges3.argtypes = [_dp] * 6 + [C.c_int64, C.c_int64, _ip]
        L.sco_eval_stat_adaptive3.argtypes = [C.POINTER(Config)] + [_dp] * 7 + [C.c_int64, C.c_int64, _ip, _dp, _ip, _dp]
        L.sco_converged.restype = C.c_int32
        L.sco_converged.argtypes = [_dp, C.c_int64, C.c_int32, C.c_double]
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ri(z):
    """complex128 array -> the same memory viewed as interleaved re/im float64."""
    if z is None:
        return None
    z = np.ascontiguousarray(z, dtype=np.complex128)
    return z.view(np.float64)


def phase(cfg, theta, f):
    th = _f64(theta)
    return lib().sco_phase(C.byref(cfg), _d(th), float(f))


def tf(cfg, theta, f):
    th = _f64(theta)
    return lib().sco_tf(C.byref(cfg), _d(th), float(f))


def phase_truth(cfg, theta, j_abs):
    """Long-double Psi at f = j_abs / T_obs -> (Psi rounded to double, remainder, cos Psi, sin Psi)."""
    th = _f64(theta)
    o = np.zeros(4)
    lib().sco_phase_truth(C.byref(cfg), _d(th), int(j_abs), _d(o))
    return o


def tf_truth(cfg, theta, j_abs):
    th = _f64(theta)
    return lib().sco_tf_truth(C.byref(cfg), _d(th), int(j_abs))


def orbit(cfg, t):
    p = np.zeros((4, 3))
    lib().sco_orbit(C.byref(cfg), float(t), _d(p))
    return p


def link(cfg, theta, f, t, s, r):
    th = _f64(theta)
    o = np.zeros(2)
    lib().sco_link(C.byref(cfg), _d(th), float(f), float(t), int(s), int(r), _d(o))
    return complex(o[0], o[1])


def tdi(cfg, theta, f, t):
    """dict X,Y,Z,A,E,T -> complex transfer function (without A(f) e^{-i Psi})."""
    th = _f64(theta)
    o = np.zeros((6, 2))
    lib().sco_tdi(C.byref(cfg), _d(th), float(f), float(t), _d(o))
    return {k: complex(o[i, 0], o[i, 1]) for i, k in enumerate("XYZAET")}


def template(cfg, theta, j_begin=0, n=None):
    """(h_A, h_E, n_in_window) on bins [j_begin, j_begin+n)."""
    n = int(cfg.n_bins - j_begin if n is None else n)
    th = _f64(theta)
    hA = np.zeros(n, dtype=np.complex128)
    hE = np.zeros(n, dtype=np.complex128)
    w = lib().sco_template(C.byref(cfg), _d(th), int(j_begin), n, _d(hA.view(np.float64)), _d(hE.view(np.float64)))
    return hA, hE, int(w)


def stat_from_arrays(dA, dE, hA, hE, SA, SE, df, edges, want_seg=False):
    edges = np.ascontiguousarray(edges, dtype=np.int64)
    n_seg = len(edges) - 1
    seg = np.zeros((n_seg, 3)) if want_seg else None
    a = [_ri(dA), _ri(dE), _ri(hA), _ri(hE), None if SA is None else _f64(SA), None if SE is None else _f64(SE)]
    u = lib().sco_stat_from_arrays(_d(a[0]), _d(a[1]), _d(a[2]), _d(a[3]), _d(a[4]), _d(a[5]), float(df),
                                   edges.ctypes.data_as(_ip), n_seg, _d(seg))
    return (u, seg) if want_seg else u


def inner(aA, aE, bA, bE, SA, SE, df):
    a = [_ri(aA), _ri(aE), _ri(bA), _ri(bE), _f64(SA), None if SE is None else _f64(SE)]
    return lib().sco_inner(_d(a[0]), _d(a[1]), _d(a[2]), _d(a[3]), _d(a[4]), _d(a[5]), float(df), len(aA))


def eval_stat(cfg, dA, dE, SA, SE, params, edges, want_seg=False, want_inwin=False):
    params = _f64(params).reshape(-1, 8)
    P = params.shape[0]
    edges = np.ascontiguousarray(edges, dtype=np.int64)
    n_seg = len(edges) - 1
    out = np.zeros(P)
    seg = np.zeros((P, n_seg, 3)) if want_seg else None
    inw = np.zeros(P, dtype=np.int64) if want_inwin else None
    a = [_ri(dA), _ri(dE), _f64(SA), _f64(SE)]
    lib().sco_eval_stat(C.byref(cfg), _d(a[0]), _d(a[1]), _d(a[2]), _d(a[3]), _d(params), P,
                        edges.ctypes.data_as(_ip), n_seg, _d(out), _d(seg),
                        None if inw is None else inw.ctypes.data_as(_ip))
    res = [out]
    if want_seg:
        res.append(seg)
    if want_inwin:
        res.append(inw)
    return res[0] if len(res) == 1 else tuple(res)


def eval_stat_levels(cfg, dA, dE, SA, SE, params, edges_list):
    """Several edge lists (hierarchy levels) from one template per particle -> [n_levels][P]."""
    params = _f64(params).reshape(-1, 8)
    P = params.shape[0]
    cat = np.ascontiguousarray(np.concatenate([np.asarray(e, dtype=np.int64) for e in edges_list]))
    ns = np.array([len(e) - 1 for e in edges_list], dtype=np.int64)
    out = np.zeros((len(edges_list), P))
    a = [_ri(dA), _ri(dE), _f64(SA), _f64(SE)]
    lib().sco_eval_stat_levels(C.byref(cfg), _d(a[0]), _d(a[1]), _d(a[2]), _d(a[3]), _d(params), P,
                               cat.ctypes.data_as(_ip), ns.ctypes.data_as(_ip), len(edges_list), _d(out))
    return out


def components_from_seg(seg, df):
    """(Upsilon_N, O_hat_N, <h|h>) from [n_seg][3] per-segment sums (Eq. 10, 8, 3)."""
    seg = _f64(seg).reshape(-1, 3)
    out = np.zeros(3)
    lib().sco_components_from_seg(_d(seg), seg.shape[0], float(df), _d(out))
    return out


def loglike(dd, hh, ohat, amp):
    return lib().sco_loglike(float(dd), float(hh), float(ohat), float(amp))


def equal_snr_edges(hA, hE, SA, SE, n_seg):
    n = len(hA)
    e = np.zeros(n_seg + 1, dtype=np.int64)
    a = [_ri(hA), None if hE is None else _ri(hE), _f64(SA), None if SE is None else _f64(SE)]
    lib().sco_equal_snr_edges(_d(a[0]), _d(a[1]), _d(a[2]), _d(a[3]), n, n_seg, e.ctypes.data_as(_ip))
    return e


def eval_stat_adaptive(cfg, dA, dE, SA, SE, params, n_seg, in_edges=None, want_edges=False, want_comp=False):
    """Upsilon_N with per-particle equal-SNR^2 edges; in_edges [P][n_seg+1] overrides the choice."""
    params = _f64(params).reshape(-1, 8)
    P = params.shape[0]
    out = np.zeros(P)
    ie = None if in_edges is None else np.ascontiguousarray(in_edges, dtype=np.int64).reshape(P, n_seg + 1)
    oe = np.zeros((P, n_seg + 1), dtype=np.int64) if want_edges else None
    oc = np.zeros((P, 3)) if want_comp else None
    a = [_ri(dA), _ri(dE), _f64(SA), _f64(SE)]
    lib().sco_eval_stat_adaptive(C.byref(cfg), _d(a[0]), _d(a[1]), _d(a[2]), _d(a[3]), _d(params), P, n_seg,
                                 None if ie is None else ie.ctypes.data_as(_ip), _d(out),
                                 None if oe is None else oe.ctypes.data_as(_ip), _d(oc))
    res = [out]
    if want_edges:
        res.append(oe)
    if want_comp:
        res.append(oc)
    return res[0] if len(res) == 1 else tuple(res)


def num_threads():
    return lib().sco_num_threads()


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) for x in key])
    o = (C.c_uint32 * 4)()
    lib().sco_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def pso_uniforms(seed, particle, it):
    rP = np.zeros(8)
    rG = np.zeros(8)
    lib().sco_pso_uniforms(int(seed), int(particle), int(it), _d(rP), _d(rG))
    return rP, rG


def pso_step(pos, vel, pbest_pos, pbest_val, stat, gbest_pos, gbest_val, lo, hi, eps_min,
             omega, phi_p, phi_g, seed, it, n_swarms):
    """In-place on float64 C-contiguous arrays (pos, vel, pbest_pos [P,8]; pbest_val [P]; gbest_* [S,8],[S])."""
    for a in (pos, vel, pbest_pos, pbest_val, gbest_pos, gbest_val):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    P = pos.shape[0]
    st, lo, hi, ep = _f64(stat), _f64(lo), _f64(hi), _f64(eps_min)
    lib().sco_pso_step(_d(pos), _d(vel), _d(pbest_pos), _d(pbest_val), _d(st), _d(gbest_pos), _d(gbest_val),
                       _d(lo), _d(hi), _d(ep), float(omega), float(phi_p), float(phi_g), int(seed), int(it),
                       P, int(n_swarms))


def pso_step_labeled(pos, vel, pbest_pos, pbest_val, stat, gbest_pos, gbest_val, label, lo, hi, eps_min,
                     omega, phi_p, phi_g, seed, it):
    """As pso_step with an int32 swarm label per particle (in place)."""
    for a in (pos, vel, pbest_pos, pbest_val, gbest_pos, gbest_val):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    lab = np.ascontiguousarray(label, dtype=np.int32)
    P, S = pos.shape[0], gbest_val.shape[0]
    st, lo, hi, ep = _f64(stat), _f64(lo), _f64(hi), _f64(eps_min)
    lib().sco_pso_step_labeled(_d(pos), _d(vel), _d(pbest_pos), _d(pbest_val), _d(st), _d(gbest_pos), _d(gbest_val),
                               lab.ctypes.data_as(C.POINTER(C.c_int32)), _d(lo), _d(hi), _d(ep), float(omega),
                               float(phi_p), float(phi_g), int(seed), int(it), P, S)


def kmeans(pos, lo, hi, cent, max_iter=100):
    """Lloyd's k-means in prior-box units -> (labels int32 [P], centroids [K,8], counts int64 [K], iterations)."""
    pos = _f64(pos).reshape(-1, 8)
    cent = np.array(cent, dtype=np.float64, order="C").reshape(-1, 8).copy()
    lo, hi = _f64(lo), _f64(hi)
    P, K = pos.shape[0], cent.shape[0]
    lab = np.zeros(P, dtype=np.int32)
    cnt = np.zeros(K, dtype=np.int64)
    it = lib().sco_kmeans(_d(pos), P, _d(lo), _d(hi), _d(cent), K, int(max_iter),
                          lab.ctypes.data_as(C.POINTER(C.c_int32)), cnt.ctypes.data_as(_ip))
    return lab, cent, cnt, int(it)


def converged(hist, window, delta):
    h = _f64(hist)
    return bool(lib().sco_converged(_d(h), len(h), int(window), float(delta)))


# ---------------------------------------------------------------------------------------------- three channels A, E, T
def template3(cfg, theta, j_begin=0, n=None):
    """(h_A, h_E, h_T, n_in_window)."""
    n = int(cfg.n_bins - j_begin if n is None else n)
    th = _f64(theta)
    h = [np.zeros(n, dtype=np.complex128) for _ in range(3)]
    w = lib().sco_template3(C.byref(cfg), _d(th), int(j_begin), n, *[_d(x.view(np.float64)) for x in h])
    return h[0], h[1], h[2], int(w)


def stat_from_arrays3(d3, h3, S3, df, edges, want_seg=False):
    """d3, h3: (A, E, T) complex arrays; S3: (S_A, S_E, S_T)."""
    edges = np.ascontiguousarray(edges, dtype=np.int64)
    n_seg = len(edges) - 1
    seg = np.zeros((n_seg, 3)) if want_seg else None
    a = [_ri(x) for x in d3] + [_ri(x) for x in h3] + [_f64(x) for x in S3]
    u = lib().sco_stat_from_arrays3(*[_d(x) for x in a], float(df), edges.ctypes.data_as(_ip), n_seg, _d(seg))
    return (u, seg) if want_seg else u


def inner3(a3, b3, S3, df):
    a = [_ri(x) for x in a3] + [_ri(x) for x in b3] + [_f64(x) for x in S3]
    return lib().sco_inner3(*[_d(x) for x in a], float(df), len(a3[0]))


def eval_stat3(cfg, d3, S3, params, edges, want_seg=False):
    params = _f64(params).reshape(-1, 8)
    P = params.shape[0]
    edges = np.ascontiguousarray(edges, dtype=np.int64)
    n_seg = len(edges) - 1
    out = np.zeros(P)
    seg = np.zeros((P, n_seg, 3)) if want_seg else None
    a = [_ri(x) for x in d3] + [_f64(x) for x in S3]
    lib().sco_eval_stat3(C.byref(cfg), *[_d(x) for x in a], _d(params), P, edges.ctypes.data_as(_ip), n_seg, _d(out), _d(seg))
    return (out, seg) if want_seg else out


def equal_snr_edges3(h3, S3, n_seg):
    """PAPER.md:120 over three channels; h3 = (hA, hE, hT) with hT possibly None (two channels)."""
    hA, hE, hT = h3
    n = len(hA)
    e = np.zeros(n_seg + 1, dtype=np.int64)
    lib().sco_equal_snr_edges3(_d(_ri(hA)), _d(_ri(hE)), None if hT is None else _d(_ri(hT)), _d(_f64(S3[0])), _d(_f64(S3[1])),
                               None if hT is None else _d(_f64(S3[2])), n, n_seg, e.ctypes.data_as(_ip))
    return e


def eval_stat_adaptive3(cfg, d3, S3, params, n_seg, in_edges=None, want_edges=False, want_comp=False):
    """Upsilon_N over A, E, T with per-particle equal-SNR^2 edges; in_edges [P][n_seg+1] overrides the choice."""
    params = _f64(params).reshape(-1, 8)
    P = params.shape[0]
    out = np.zeros(P)
    ie = None if in_edges is None else np.ascontiguousarray(in_edges, dtype=np.int64).reshape(P, n_seg + 1)
    oe = np.zeros((P, n_seg + 1), dtype=np.int64) if want_edges else None
    oc = np.zeros((P, 3)) if want_comp else None
    a = [_ri(x) for x in d3] + [_f64(x) for x in S3]
    lib().sco_eval_stat_adaptive3(C.byref(cfg), *[_d(x) for x in a], _d(params), P, n_seg,
                                  None if ie is None else ie.ctypes.data_as(_ip), _d(out),
                                  None if oe is None else oe.ctypes.data_as(_ip), _d(oc))
    res = [out]
    if want_edges:
        res.append(oe)
    if want_comp:
        res.append(oc)
    return res[0] if len(res) == 1 else tuple(res)
