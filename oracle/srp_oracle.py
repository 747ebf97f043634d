"""ctypes front end of the CPU oracle -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  The product
(``paper_2602_10712_b200``) never does, and this module imports nothing from it.

The arithmetic lives in ``srp_oracle_mesh.c`` / ``srp_oracle_trace.c`` (fp64, single
thread, brute force over all triangles -- PAPER.md:159).  This file only compiles
them with gcc and marshals numpy arrays.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SOURCES = ["srp_oracle_mesh.c", "srp_oracle_trace.c"]
_LIB_PATH = os.path.join(_HERE, "libsrp_oracle.so")

FAMILY_PLATE, FAMILY_BOXWING, FAMILY_DETAILED, FAMILY_BOXWING6, FAMILY_SAIL, FAMILY_BOXWING_T = range(6)
SOLAR_PRESSURE = 4.56e-6  # N/m^2 at 1 AU (BASELINE.json config 1)


class Stats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_ulonglong) for n in
                ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments")] + \
               [("hits_at_depth", ctypes.c_ulonglong * 16)]

    def as_dict(self):
        d = {n: int(getattr(self, n)) for n, _ in self._fields_[:6]}
        d["hits_at_depth"] = [int(x) for x in self.hits_at_depth]
        return d


class Options(ctypes.Structure):
    _fields_ = [("solar_pressure", ctypes.c_double), ("sampler", ctypes.c_int),
                ("deposit", ctypes.c_int), ("no_caustics", ctypes.c_int)]


def build(force=False):
    """Compile the oracle's C sources into oracle/libsrp_oracle.so (gcc, -O2, no FMA contraction)."""
    srcs = [os.path.join(_HERE, s) for s in _SOURCES]
    deps = srcs + [os.path.join(_HERE, "srp_oracle_common.h")]
    if (not force and os.path.exists(_LIB_PATH)
            and all(os.path.getmtime(_LIB_PATH) >= os.path.getmtime(d) for d in deps)):
        return _LIB_PATH
    tmp = _LIB_PATH + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-std=c99", "-Wall", "-fPIC", "-shared",
           *srcs, "-o", tmp, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB_PATH)
    return _LIB_PATH


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.srp_oracle_n_params.restype = ctypes.c_int
        L.srp_oracle_n_params.argtypes = [ctypes.c_int]
        L.srp_oracle_tri_count.restype = ctypes.c_long
        L.srp_oracle_tri_count.argtypes = [ctypes.c_int]
        L.srp_oracle_build_mesh.restype = ctypes.c_long
        L.srp_oracle_build_mesh.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_int,
                                            ctypes.c_uint64, ctypes.c_void_p, ctypes.c_void_p]
        L.srp_oracle_forces.restype = ctypes.c_int
        L.srp_oracle_forces.argtypes = [
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_long, ctypes.c_int,
            ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_longlong, ctypes.c_int,
            ctypes.c_ulonglong, ctypes.POINTER(Options),
            ctypes.c_void_p, ctypes.c_void_p, ctypes.POINTER(Stats), ctypes.c_void_p, ctypes.c_void_p]
        L.srp_oracle_forces_torques.restype = ctypes.c_int
        L.srp_oracle_forces_torques.argtypes = L.srp_oracle_forces.argtypes + [ctypes.c_void_p] * 3
        L.srp_oracle_forces_torques_glossy.restype = ctypes.c_int
        a = L.srp_oracle_forces_torques.argtypes
        L.srp_oracle_forces_torques_glossy.argtypes = a[:2] + [ctypes.c_void_p] + a[2:]
        L.srp_oracle_forces_split.restype = ctypes.c_int
        L.srp_oracle_forces_split.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_long, ctypes.c_int,
                                              ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_longlong, ctypes.c_int,
                                              ctypes.c_ulonglong, ctypes.POINTER(Options), ctypes.c_void_p, ctypes.c_void_p,
                                              ctypes.POINTER(Stats)]
        L.srp_oracle_backward.restype = ctypes.c_int
        L.srp_oracle_backward.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_long, ctypes.c_int, ctypes.c_void_p,
                                          ctypes.c_int, ctypes.c_longlong, ctypes.c_int, ctypes.c_ulonglong,
                                          ctypes.POINTER(Options), ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        L.srp_oracle_thermal.restype = ctypes.c_int
        L.srp_oracle_thermal.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_long, ctypes.c_int, ctypes.c_void_p,
                                         ctypes.c_longlong, ctypes.c_int, ctypes.c_ulonglong, ctypes.POINTER(Options),
                                         ctypes.c_void_p, ctypes.c_void_p, ctypes.POINTER(Stats)]
        L.srp_oracle_thermal_glossy.restype = ctypes.c_int
        a = L.srp_oracle_thermal.argtypes
        L.srp_oracle_thermal_glossy.argtypes = a[:2] + [ctypes.c_void_p] + a[2:]
        L.srp_oracle_sail_height.restype = ctypes.c_double
        L.srp_oracle_sail_height.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_uint64]
        L.srp_oracle_philox.restype = None
        L.srp_oracle_philox.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        L.srp_oracle_uniform.restype = ctypes.c_double
        L.srp_oracle_uniform.argtypes = [ctypes.c_uint32]
        _lib = L
    return _lib


def philox(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().srp_oracle_philox(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out


def uniform(x):
    return lib().srp_oracle_uniform(int(x) & 0xFFFFFFFF)


def sail_height(x, y, amp=0.05, mesh_seed=2):
    """Height of the SAIL family's noise surface above (x, y)."""
    return lib().srp_oracle_sail_height(float(x), float(y), float(amp), int(mesh_seed))


def n_params(family):
    return lib().srp_oracle_n_params(family)


def tri_count(family):
    return lib().srp_oracle_tri_count(family)


def build_mesh(family, theta, k=0, mesh_seed=2):
    """Mesh of ONE design: theta float32[n_params]; returns (verts f32[T,3,3], mats f32[T,3])."""
    theta = np.ascontiguousarray(theta, dtype=np.float32).reshape(-1)
    if theta.size != n_params(family):
        raise ValueError("family %d takes %d parameters" % (family, n_params(family)))
    T = tri_count(family)
    verts = np.empty((T, 3, 3), dtype=np.float32)
    mats = np.empty((T, 3), dtype=np.float32)
    got = lib().srp_oracle_build_mesh(family, theta.ctypes.data, int(k), int(mesh_seed),
                                      verts.ctypes.data, mats.ctypes.data)
    if got != T:
        raise RuntimeError("oracle mesh build failed")
    return verts, mats


def forces(verts, mats, sun_dirs, N, B, seed=0, k=0, j0=0, P=SOLAR_PRESSURE, sampler=0,
           deposit=0, want_first_hit=False, want_path_sig=False, x_com=None, shininess=None, no_caustics=0):
    """Forces of ONE design for the given sun directions.

    Returns dict(F f64[S,3], sumsq f64[S,3], sigma f64[S] (i.i.d. standard error of |F|,
    conservative for the stratified sampler), stats dict, first_hit int32[S,N] or None).
    With x_com (3 floats, the centre of mass of PAPER.md:136 Eq. 4) also T f64[S,3] (torque, N m)
    and sigma_T f64[S].  shininess float32[T]: Phong exponent of each facet's specular lobe, < 0 = ideal mirror
    (R23); None = ideal mirrors throughout.
    """
    verts = np.ascontiguousarray(verts, dtype=np.float32).reshape(-1, 3, 3)
    mats = np.ascontiguousarray(mats, dtype=np.float32).reshape(-1, 3)
    sun = np.ascontiguousarray(sun_dirs, dtype=np.float32).reshape(-1, 3)
    T, S = verts.shape[0], sun.shape[0]
    assert mats.shape[0] == T
    F = np.zeros((S, 3)); Q = np.zeros((S, 3))
    st = Stats()
    fh = np.empty((S, N), dtype=np.int32) if want_first_hit else None
    ps = np.empty((S, N), dtype=np.uint64) if want_path_sig else None
    opt = Options(float(P), int(sampler), int(deposit), int(no_caustics))
    args = (verts.ctypes.data, mats.ctypes.data, T, int(k), sun.ctypes.data,
            S, int(j0), int(N), int(B), int(seed), ctypes.byref(opt),
            F.ctypes.data, Q.ctypes.data, ctypes.byref(st),
            fh.ctypes.data if fh is not None else None,
            ps.ctypes.data if ps is not None else None)
    Tq = TQ = None
    if shininess is not None:
        sh = np.ascontiguousarray(shininess, dtype=np.float32).reshape(-1)
        assert sh.shape[0] == T
        xc = None if x_com is None else np.ascontiguousarray(x_com, dtype=np.float64).reshape(3)
        if xc is not None:
            Tq = np.zeros((S, 3)); TQ = np.zeros((S, 3))
        rc = lib().srp_oracle_forces_torques_glossy(*args[:2], sh.ctypes.data, *args[2:],
                                                    xc.ctypes.data if xc is not None else None,
                                                    Tq.ctypes.data if xc is not None else None,
                                                    TQ.ctypes.data if xc is not None else None)
    elif x_com is None:
        rc = lib().srp_oracle_forces(*args)
    else:
        xc = np.ascontiguousarray(x_com, dtype=np.float64).reshape(3)
        Tq = np.zeros((S, 3)); TQ = np.zeros((S, 3))
        rc = lib().srp_oracle_forces_torques(*args, xc.ctypes.data, Tq.ctypes.data, TQ.ctypes.data)
    if rc != 0:
        raise ValueError("srp_oracle_forces: invalid arguments")
    var = np.maximum(Q - F * F / float(N), 0.0)     # N * sample variance of the photon totals
    sigma = np.sqrt(var.sum(axis=1))
    out = {"F": F, "sumsq": Q, "sigma": sigma, "stats": st.as_dict(), "first_hit": fh, "path_sig": ps}
    if Tq is not None:
        out["T"] = Tq
        out["sigma_T"] = np.sqrt(np.maximum(TQ - Tq * Tq / float(N), 0.0).sum(axis=1))
    return out


def forces_split(verts, mats, sun_dirs, N, B, seed=0, k=0, j0=0, P=SOLAR_PRESSURE, sampler=0, deposit=0, shininess=None):
    """Total force and its direct part (momentum deposited where sun light first meets the surface)
    Fig. 5: dict(F f64[S,3], F_direct f64[S,3], F_indirect = F - F_direct, stats)."""
    verts = np.ascontiguousarray(verts, dtype=np.float32).reshape(-1, 3, 3)
    mats = np.ascontiguousarray(mats, dtype=np.float32).reshape(-1, 3)
    sun = np.ascontiguousarray(sun_dirs, dtype=np.float32).reshape(-1, 3)
    T, S = verts.shape[0], sun.shape[0]
    sh = None if shininess is None else np.ascontiguousarray(shininess, dtype=np.float32).reshape(-1)
    F = np.zeros((S, 3)); Fd = np.zeros((S, 3))
    st = Stats()
    opt = Options(float(P), int(sampler), int(deposit), 0)
    rc = lib().srp_oracle_forces_split(verts.ctypes.data, mats.ctypes.data, sh.ctypes.data if sh is not None else None, T,
                                       int(k), sun.ctypes.data, S, int(j0), int(N), int(B), int(seed), ctypes.byref(opt),
                                       F.ctypes.data, Fd.ctypes.data, ctypes.byref(st))
    if rc != 0:
        raise ValueError("srp_oracle_forces_split: invalid arguments")
    return {"F": F, "F_direct": Fd, "F_indirect": F - Fd, "stats": st.as_dict()}


def backward(verts, mats, sun_dir, N, B, seed=0, k=0, j=0, P=SOLAR_PRESSURE, deposit=0):
    """The paper's backward estimator (Eq. 5) of ONE (design, direction) pair: N surface samples,
    paths of at most B vertices with next-event estimation.  A cross-check of `forces`.  Returns dict(F f64[3],
    sigma (standard error of |F|), n_nee)."""
    verts = np.ascontiguousarray(verts, dtype=np.float32).reshape(-1, 3, 3)
    mats = np.ascontiguousarray(mats, dtype=np.float32).reshape(-1, 3)
    w = np.ascontiguousarray(sun_dir, dtype=np.float32).reshape(3)
    F = np.zeros(3); Q = np.zeros(3)
    nee = ctypes.c_ulonglong()
    opt = Options(float(P), 1, int(deposit), 0)
    rc = lib().srp_oracle_backward(verts.ctypes.data, mats.ctypes.data, verts.shape[0], int(k), w.ctypes.data, int(j),
                                   int(N), int(B), int(seed), ctypes.byref(opt), F.ctypes.data, Q.ctypes.data,
                                   ctypes.byref(nee))
    if rc != 0:
        raise ValueError("srp_oracle_backward: invalid arguments")
    var = np.maximum(Q / N - F * F, 0.0) / N             # variance of the mean of the per-sample totals
    return {"F": F, "sigma": float(np.sqrt(var.sum())), "n_nee": int(nee.value)}


def thermal(verts, mats, facet_power, N, B, seed=0, k=0, deposit=0, shininess=None):
    """Recoil force of ONE design's thermal (Lambertian) facet emitters: facet_power float32[T]
    in watts, signed (sign = emitting side), N photons per emitting facet.  Returns dict(F f64[3] newtons,
    sigma f64 (i.i.d. standard error of |F| over all emitted photons), stats)."""
    verts = np.ascontiguousarray(verts, dtype=np.float32).reshape(-1, 3, 3)
    mats = np.ascontiguousarray(mats, dtype=np.float32).reshape(-1, 3)
    pw = np.ascontiguousarray(facet_power, dtype=np.float32).reshape(-1)
    T = verts.shape[0]
    assert mats.shape[0] == T and pw.shape[0] == T
    F = np.zeros(3); Q = np.zeros(3)
    st = Stats()
    opt = Options(float(SOLAR_PRESSURE), 0, int(deposit), 0)
    sh = None if shininess is None else np.ascontiguousarray(shininess, dtype=np.float32).reshape(-1)
    assert sh is None or sh.shape[0] == T
    rc = lib().srp_oracle_thermal_glossy(verts.ctypes.data, mats.ctypes.data, sh.ctypes.data if sh is not None else None,
                                         T, int(k), pw.ctypes.data, int(N), int(B),
                                         int(seed), ctypes.byref(opt), F.ctypes.data, Q.ctypes.data, ctypes.byref(st))
    if rc != 0:
        raise ValueError("srp_oracle_thermal: invalid arguments")
    n = max(int(st.launched), 1)
    sigma = float(np.sqrt(np.maximum(Q - F * F / n, 0.0).sum()))
    return {"F": F, "sigma": sigma, "stats": st.as_dict()}
