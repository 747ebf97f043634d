"""Thin Python binding of the C ABI in include/srp.h (same names, argument marshalling only).

PyTorch supplies device memory (tensors) and the CUDA stream; every step of the path runs in the
library's kernels.  There is no fallback: if ``libsrp_b200.so`` is missing or no CUDA device is
present, calls raise.
"""
import ctypes
import os

import numpy as np
import torch

from . import workloads as W

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsrp_b200.so")

SRP_OK = 0
_STATUS = {0: "SRP_OK", -1: "SRP_ERR_INVALID", -2: "SRP_ERR_CUDA", -3: "SRP_ERR_OOM", -4: "SRP_ERR_UNSUPPORTED"}


class SrpError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("%s: %s" % (_STATUS.get(status, status), text))
        self.status = status


class srp_options(ctypes.Structure):
    _fields_ = [("solar_pressure", ctypes.c_double), ("sampler", ctypes.c_int), ("deposit", ctypes.c_int),
                ("force_brute", ctypes.c_int), ("instrumented", ctypes.c_int), ("primary_mode", ctypes.c_int), ("escape_masks", ctypes.c_int),
                ("plain_launches", ctypes.c_int), ("leaf_max", ctypes.c_int),
                ("bvh_builder", ctypes.c_int)]


class srp_stats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_ulonglong) for n in
                ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments")] + \
               [("hits_at_depth", ctypes.c_ulonglong * 16), ("box_tests", ctypes.c_ulonglong),
                ("tri_tests", ctypes.c_ulonglong)] + \
               [(n, ctypes.c_ulonglong) for n in ("beam_tile_miss", "beam_block_miss", "beam_group_miss", "beam_fallback",
                                                  "beam_box_tests", "tri2d_tests", "tri_setups", "rect_tests", "mask_escapes",
                                                  "queued_rays", "loop_rounds", "kernel_launches")]

    def as_dict(self):
        d = {n: int(getattr(self, n)) for n in
             ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments", "box_tests", "tri_tests",
              "beam_tile_miss", "beam_block_miss", "beam_group_miss", "beam_fallback",
              "beam_box_tests", "tri2d_tests", "tri_setups", "rect_tests", "mask_escapes", "queued_rays", "loop_rounds",
              "kernel_launches")}
        d["hits_at_depth"] = [int(x) for x in self.hits_at_depth]
        return d


EXPORTS = ["srp_create", "srp_destroy", "srp_set_options", "srp_get_options", "srp_last_error",
           "srp_family_n_params", "srp_family_tri_count", "srp_build_designs",
           "srp_build_designs_from_meshes", "srp_designs_info", "srp_designs_read_mesh",
           "srp_designs_read_bvh", "srp_free_designs", "srp_forces", "srp_forces_pairs", "srp_forces_host",
           "srp_forces_torques", "srp_forces_torques_pairs", "srp_forces_split", "srp_forces_split_pairs",
           "srp_forces_per_sample", "srp_forces_noalloc", "srp_thermal_forces", "srp_designs_set_shininess", "srp_first_hits", "srp_path_signatures", "srp_get_stats",
           "srp_launch_count", "srp_set_workspace", "srp_workspace_bytes_min", "srp_probe_peaks"]

_lib = None


def load_library():
    """dlopen libsrp_b200.so and declare the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libsrp_b200.so is not built: run `python -m paper_2602_10712_b200.build` "
                           "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, ci, ll, ull = ctypes.c_void_p, ctypes.c_int, ctypes.c_longlong, ctypes.c_ulonglong
    L.srp_create.argtypes = [ctypes.POINTER(vp), ci, vp]
    L.srp_destroy.argtypes = [vp]
    L.srp_set_options.argtypes = [vp, ctypes.POINTER(srp_options)]
    L.srp_get_options.argtypes = [vp, ctypes.POINTER(srp_options)]
    L.srp_last_error.argtypes = [vp]
    L.srp_last_error.restype = ctypes.c_char_p
    L.srp_family_n_params.argtypes = [ci]
    L.srp_family_tri_count.argtypes = [ci]
    L.srp_family_tri_count.restype = ll
    L.srp_build_designs.argtypes = [vp, ci, vp, ci, ci, ull, ctypes.POINTER(vp)]
    L.srp_build_designs_from_meshes.argtypes = [vp, vp, vp, vp, ci, ctypes.POINTER(vp)]
    L.srp_designs_info.argtypes = [vp, ctypes.POINTER(ci), vp]
    L.srp_designs_read_mesh.argtypes = [vp, vp, ci, vp, vp]
    L.srp_designs_read_bvh.argtypes = [vp, vp, ci, ctypes.POINTER(ll), vp, vp]
    L.srp_free_designs.argtypes = [vp, vp]
    L.srp_forces.argtypes = [vp, vp, vp, ci, ll, ci, ull, vp]
    L.srp_forces_noalloc.argtypes = [vp, vp, vp, ci, ll, ci, ull, vp]
    L.srp_forces_pairs.argtypes = [vp, vp, vp, ci, vp, ll, ll, ci, ull, vp]
    L.srp_forces_host.argtypes = [vp, vp, vp, ci, ll, ci, ull, vp]
    L.srp_forces_torques.argtypes = [vp, vp, vp, ci, ll, ci, ull, vp, vp, vp]
    L.srp_forces_torques_pairs.argtypes = [vp, vp, vp, ci, vp, ll, ll, ci, ull, vp, vp, vp]
    L.srp_forces_split.argtypes = [vp, vp, vp, ci, ll, ci, ull, vp, vp]
    L.srp_forces_split_pairs.argtypes = [vp, vp, vp, ci, vp, ll, ll, ci, ull, vp, vp]
    L.srp_forces_per_sample.argtypes = [vp, ci, vp, ci, vp, ll, ll, ci, ull, ull, vp]
    L.srp_launch_count.argtypes = [vp, ctypes.POINTER(ull)]
    L.srp_set_workspace.argtypes = [vp, vp, ull]
    L.srp_workspace_bytes_min.argtypes = [vp]
    L.srp_workspace_bytes_min.restype = ull
    L.srp_thermal_forces.argtypes = [vp, vp, vp, ll, ci, ull, vp]
    L.srp_designs_set_shininess.argtypes = [vp, vp, vp]
    L.srp_first_hits.argtypes = [vp, vp, vp, ci, vp, ll, ll, ull, ci, vp]
    L.srp_path_signatures.argtypes = [vp, vp, vp, ci, vp, ll, ll, ci, ull, vp]
    L.srp_get_stats.argtypes = [vp, ctypes.POINTER(srp_stats)]
    L.srp_probe_peaks.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    for name in EXPORTS:
        if name not in ("srp_last_error", "srp_family_tri_count", "srp_workspace_bytes_min"):
            getattr(L, name).restype = ci
    _lib = L
    return L


def _f32_cuda(t, device):
    t = torch.as_tensor(t)
    return t.to(device=device, dtype=torch.float32).contiguous()


def _check_cuda_f32(t, name, device, shape_tail=None):
    """A contiguous float32 CUDA tensor on `device` (its data_ptr() is handed to the library as a DEVICE pointer)."""
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.device == device and t.dtype == torch.float32 and t.is_contiguous()):
        raise ValueError("%s must be a contiguous float32 CUDA tensor on %s" % (name, device))
    if shape_tail is not None and tuple(t.shape[-len(shape_tail):]) != tuple(shape_tail):
        raise ValueError("%s must have shape [..., %s]" % (name, ", ".join(map(str, shape_tail))))
    return t


class Designs:
    """Owner of an ``srp_designs*`` handle."""

    def __init__(self, ctx, handle):
        self.ctx, self.handle = ctx, handle
        D = ctypes.c_int()
        ctx._check(ctx.lib.srp_designs_info(handle, ctypes.byref(D), None))
        self.D = D.value
        off = np.zeros(self.D + 1, dtype=np.int64)
        ctx._check(ctx.lib.srp_designs_info(handle, None, off.ctypes.data))
        self.tri_offsets = off

    def read_mesh(self, design):
        T = int(self.tri_offsets[design + 1] - self.tri_offsets[design])
        v = np.empty((T, 3, 3), np.float32)
        m = np.empty((T, 3), np.float32)
        self.ctx._check(self.ctx.lib.srp_designs_read_mesh(self.ctx.handle, self.handle, design,
                                                           v.ctypes.data, m.ctypes.data))
        return v, m

    def read_bvh(self, design):
        n = ctypes.c_longlong()
        T = int(self.tri_offsets[design + 1] - self.tri_offsets[design])
        self.ctx._check(self.ctx.lib.srp_designs_read_bvh(self.ctx.handle, self.handle, design,
                                                          ctypes.byref(n), None, None))
        nodes = np.empty((n.value, 16), np.float32)
        perm = np.empty(T, np.int32)
        self.ctx._check(self.ctx.lib.srp_designs_read_bvh(self.ctx.handle, self.handle, design, ctypes.byref(n),
                                                          nodes.ctypes.data if n.value else None, perm.ctypes.data))
        return nodes, perm

    def free(self):
        if self.handle:
            self.ctx.lib.srp_free_designs(self.ctx.handle, self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Context:
    """Owner of an ``srp_context*``; work is enqueued on torch's current stream of `device` at creation."""

    def __init__(self, device=0, stream=None):
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: libsrp_b200 has no CPU fallback")
        self.lib = load_library()
        self.device = torch.device("cuda", device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = ctypes.c_void_p()
        st = self.lib.srp_create(ctypes.byref(h), device, ctypes.c_void_p(self.stream.cuda_stream))
        if st != SRP_OK:
            raise SrpError(st, "srp_create failed")
        self.handle = h

    def _check(self, st):
        if st != SRP_OK:
            raise SrpError(st, self.lib.srp_last_error(self.handle).decode())

    def close(self):
        if self.handle:
            self.lib.srp_destroy(self.handle)
            self.handle = None

    def srp_set_options(self, solar_pressure=W.SOLAR_PRESSURE, sampler=0, deposit=0, force_brute=0, instrumented=0,
                        primary_mode=0, escape_masks=1, plain_launches=0, leaf_max=0, bvh_builder=0):
        o = srp_options(solar_pressure, sampler, deposit, force_brute, instrumented, primary_mode, escape_masks,
                        plain_launches, leaf_max, bvh_builder)
        self._check(self.lib.srp_set_options(self.handle, ctypes.byref(o)))

    def srp_build_designs(self, family, theta, mesh_seed=W.MESH_SEED):
        theta = _f32_cuda(theta, self.device)
        if theta.dim() != 2:
            raise ValueError("theta must be [D, n_params]")
        h = ctypes.c_void_p()
        self._check(self.lib.srp_build_designs(self.handle, family, theta.data_ptr(), theta.shape[0],
                                               theta.shape[1], mesh_seed, ctypes.byref(h)))
        self.stream.synchronize()          # theta may be a temporary
        return Designs(self, h)

    def srp_build_designs_from_meshes(self, verts, mats, tri_offsets):
        if isinstance(mats, np.ndarray):           # host data: check what the header asks of the materials
            m = np.asarray(mats, np.float64).reshape(-1, 3)
            if not (np.all(m >= 0.0) and np.all(np.abs(m.sum(1) - 1.0) <= 1e-5)):
                raise ValueError("materials must be >= 0 and sum to 1 per facet")
        verts, mats = _f32_cuda(verts, self.device), _f32_cuda(mats, self.device)
        off = np.ascontiguousarray(tri_offsets, dtype=np.int64)
        if verts.numel() != 9 * int(off[-1]) or mats.numel() != 3 * int(off[-1]):
            raise ValueError("verts / mats do not match tri_offsets")
        h = ctypes.c_void_p()
        self._check(self.lib.srp_build_designs_from_meshes(self.handle, verts.data_ptr(), mats.data_ptr(),
                                                           off.ctypes.data, len(off) - 1, ctypes.byref(h)))
        self.stream.synchronize()
        return Designs(self, h)

    def srp_forces_noalloc(self, designs, sun_dirs, rays_per_dir, max_bounces, seed, out):
        """srp_forces through the library's static scratch: allocates nothing (the caller brings `out`, CUDA float32
        [D,S,3]); at most NOALLOC_MAX_PAIRS (design, direction) pairs, no beam-traced calls (include/srp.h)."""
        _check_cuda_f32(sun_dirs, "sun_dirs", self.device, (3,))
        S = sun_dirs.shape[0]
        if _check_cuda_f32(out, "out", self.device).numel() != designs.D * S * 3:
            raise ValueError("out must hold [D, S, 3] floats")
        self._check(self.lib.srp_forces_noalloc(self.handle, designs.handle, sun_dirs.data_ptr(), S, rays_per_dir,
                                                max_bounces, seed, out.data_ptr()))
        return out

    def srp_forces(self, designs, sun_dirs, rays_per_dir, max_bounces, seed=0, out=None):
        """sun_dirs: CUDA float32 [S,3]; returns CUDA float32 [D,S,3] (asynchronous on the stream)."""
        _check_cuda_f32(sun_dirs, "sun_dirs", self.device, (3,))
        S = sun_dirs.shape[0]
        if out is None:
            out = torch.empty((designs.D, S, 3), dtype=torch.float32, device=self.device)
        elif _check_cuda_f32(out, "out", self.device).numel() != designs.D * S * 3:
            raise ValueError("out must hold [D, S, 3] floats")
        self._check(self.lib.srp_forces(self.handle, designs.handle, sun_dirs.data_ptr(), S, rays_per_dir,
                                        max_bounces, seed, out.data_ptr()))
        return out

    def _pairs(self, designs, sun_dirs, pairs):
        _check_cuda_f32(sun_dirs, "sun_dirs", self.device, (3,))
        pairs = torch.as_tensor(pairs).to(device=self.device, dtype=torch.int32).contiguous()
        if pairs.dim() != 2 or pairs.shape[1] != 2 or pairs.shape[0] == 0:
            raise ValueError("pairs must be [n, 2]")
        lo, hi = pairs.min(0).values.tolist(), pairs.max(0).values.tolist()
        if lo[0] < 0 or lo[1] < 0 or hi[0] >= designs.D or hi[1] >= sun_dirs.shape[0]:
            raise ValueError("pairs out of range")
        return pairs

    def srp_forces_pairs(self, designs, sun_dirs, pairs, rays_per_dir, max_bounces, seed=0):
        pairs = self._pairs(designs, sun_dirs, pairs)
        out = torch.empty((pairs.shape[0], 3), dtype=torch.float32, device=self.device)
        self._check(self.lib.srp_forces_pairs(self.handle, designs.handle, sun_dirs.data_ptr(), sun_dirs.shape[0],
                                              pairs.data_ptr(), pairs.shape[0], rays_per_dir, max_bounces, seed,
                                              out.data_ptr()))
        self.stream.synchronize()
        return out

    def _xcom(self, designs, x_com):
        if x_com is None:
            return None
        x = torch.as_tensor(x_com).to(device=self.device, dtype=torch.float32).contiguous()
        if tuple(x.shape) != (designs.D, 3):
            raise ValueError("x_com must be [D, 3]")
        return x

    def srp_forces_torques(self, designs, sun_dirs, rays_per_dir, max_bounces, seed=0, x_com=None):
        """Forces and torques about x_com ([D,3], None = origin): two CUDA float32 [D,S,3] tensors."""
        _check_cuda_f32(sun_dirs, "sun_dirs", self.device, (3,))
        S = sun_dirs.shape[0]
        x = self._xcom(designs, x_com)
        F = torch.empty((designs.D, S, 3), dtype=torch.float32, device=self.device)
        T = torch.empty((designs.D, S, 3), dtype=torch.float32, device=self.device)
        self._check(self.lib.srp_forces_torques(self.handle, designs.handle, sun_dirs.data_ptr(), S, rays_per_dir,
                                                max_bounces, seed, x.data_ptr() if x is not None else None,
                                                F.data_ptr(), T.data_ptr()))
        self.stream.synchronize()
        return F, T

    def srp_forces_torques_pairs(self, designs, sun_dirs, pairs, rays_per_dir, max_bounces, seed=0, x_com=None):
        pairs = self._pairs(designs, sun_dirs, pairs)
        x = self._xcom(designs, x_com)
        F = torch.empty((pairs.shape[0], 3), dtype=torch.float32, device=self.device)
        T = torch.empty((pairs.shape[0], 3), dtype=torch.float32, device=self.device)
        self._check(self.lib.srp_forces_torques_pairs(self.handle, designs.handle, sun_dirs.data_ptr(),
                                                      sun_dirs.shape[0], pairs.data_ptr(), pairs.shape[0],
                                                      rays_per_dir, max_bounces, seed,
                                                      x.data_ptr() if x is not None else None, F.data_ptr(),
                                                      T.data_ptr()))
        self.stream.synchronize()
        return F, T

    def srp_designs_set_shininess(self, designs, shininess):
        """shininess: float32 [sumT] Phong exponents in original triangle order (< 0 = ideal mirror), or None to
        remove them (R23)."""
        if shininess is None:
            self._check(self.lib.srp_designs_set_shininess(self.handle, designs.handle, None))
            return
        sh = torch.as_tensor(shininess).to(device=self.device, dtype=torch.float32).contiguous()
        if sh.numel() != int(designs.tri_offsets[-1]):
            raise ValueError("shininess must have one entry per triangle of the batch")
        self._check(self.lib.srp_designs_set_shininess(self.handle, designs.handle, sh.data_ptr()))
        self.stream.synchronize()          # sh may be a temporary

    def srp_thermal_forces(self, designs, facet_power, rays_per_facet, max_bounces, seed=0):
        """facet_power: float32 [sumT] watts in original triangle order (signed: emitting side); returns CUDA
        float32 [D,3] recoil forces in newtons."""
        pw = torch.as_tensor(facet_power).to(device=self.device, dtype=torch.float32).contiguous()
        if pw.numel() != int(designs.tri_offsets[-1]):
            raise ValueError("facet_power must have one entry per triangle of the batch")
        out = torch.empty((designs.D, 3), dtype=torch.float32, device=self.device)
        self._check(self.lib.srp_thermal_forces(self.handle, designs.handle, pw.data_ptr(), rays_per_facet, max_bounces,
                                                seed, out.data_ptr()))
        self.stream.synchronize()
        return out

    def srp_forces_split(self, designs, sun_dirs, rays_per_dir, max_bounces, seed=0):
        """Forces and their direct part (momentum deposited where sun light first meets the surface)
        from one trace: two CUDA float32 [D,S,3] tensors (asynchronous on the stream)."""
        _check_cuda_f32(sun_dirs, "sun_dirs", self.device, (3,))
        S = sun_dirs.shape[0]
        F = torch.empty((designs.D, S, 3), dtype=torch.float32, device=self.device)
        Fd = torch.empty((designs.D, S, 3), dtype=torch.float32, device=self.device)
        self._check(self.lib.srp_forces_split(self.handle, designs.handle, sun_dirs.data_ptr(), S, rays_per_dir,
                                              max_bounces, seed, F.data_ptr(), Fd.data_ptr()))
        return F, Fd

    def srp_forces_split_pairs(self, designs, sun_dirs, pairs, rays_per_dir, max_bounces, seed=0):
        pairs = self._pairs(designs, sun_dirs, pairs)
        F = torch.empty((pairs.shape[0], 3), dtype=torch.float32, device=self.device)
        Fd = torch.empty((pairs.shape[0], 3), dtype=torch.float32, device=self.device)
        self._check(self.lib.srp_forces_split_pairs(self.handle, designs.handle, sun_dirs.data_ptr(), sun_dirs.shape[0],
                                                    pairs.data_ptr(), pairs.shape[0], rays_per_dir, max_bounces, seed,
                                                    F.data_ptr(), Fd.data_ptr()))
        self.stream.synchronize()
        return F, Fd

    def srp_forces_per_sample(self, family, theta, sun_dirs, rays_per_record, max_bounces, seed=0, mesh_seed=W.MESH_SEED,
                              out=None):
        """The paper's workload shape: record m = its own design theta[m] lit from its own
        direction sun_dirs[m].  theta [M, n_params], sun_dirs [M, 3] (CUDA float32); returns CUDA float32 [M, 3]
        (asynchronous on the stream)."""
        _check_cuda_f32(theta, "theta", self.device)
        _check_cuda_f32(sun_dirs, "sun_dirs", self.device, (3,))
        M = theta.shape[0]
        if theta.dim() != 2 or sun_dirs.shape[0] != M:
            raise ValueError("theta must be [M, n_params] and sun_dirs [M, 3]")
        if out is None:
            out = torch.empty((M, 3), dtype=torch.float32, device=self.device)
        elif _check_cuda_f32(out, "out", self.device).numel() != 3 * M:
            raise ValueError("out must hold [M, 3] floats")
        self._check(self.lib.srp_forces_per_sample(self.handle, family, theta.data_ptr(), theta.shape[1], sun_dirs.data_ptr(),
                                                   M, rays_per_record, max_bounces, seed, mesh_seed, out.data_ptr()))
        return out

    def force_maps(self, designs, n_lat, n_lon, rays_per_dir, max_bounces, seed=0):
        """The paper's force-map figures (Fig. 5): forces over a latitude-longitude image of sun
        directions (workloads.latlong_directions) with their direct part, from one srp_forces_split call, reshaped:
        two CUDA float32 [D, n_lat, n_lon, 3] tensors (total, direct); the indirect map is their difference."""
        sun = torch.from_numpy(W.latlong_directions(n_lat, n_lon)).to(self.device)
        total, direct = self.srp_forces_split(designs, sun, rays_per_dir, max_bounces, seed)
        shape = (designs.D, n_lat, n_lon, 3)
        return total.reshape(shape), direct.reshape(shape)

    def srp_set_workspace(self, tensor):
        """Hands the library a CUDA tensor (any dtype, contiguous) as the ray queue of its beam / bounce loop, or
        None to let it allocate its own.  The tensor is kept alive by this object."""
        if tensor is None:
            self._check(self.lib.srp_set_workspace(self.handle, None, 0))
        else:
            if not (tensor.is_cuda and tensor.device == self.device and tensor.is_contiguous()):
                raise ValueError("workspace must be a contiguous CUDA tensor on %s" % self.device)
            self._check(self.lib.srp_set_workspace(self.handle, tensor.data_ptr(), tensor.numel() * tensor.element_size()))
        self._workspace = tensor

    def srp_workspace_bytes_min(self):
        return int(self.lib.srp_workspace_bytes_min(self.handle))

    def srp_launch_count(self):
        n = ctypes.c_ulonglong()
        self._check(self.lib.srp_launch_count(self.handle, ctypes.byref(n)))
        return n.value

    def srp_forces_host(self, designs, sun_dirs_host, rays_per_dir, max_bounces, seed=0, out_host=None):
        """Host buffers in and out (numpy float32 or pinned CPU tensors); synchronous."""
        s = sun_dirs_host if isinstance(sun_dirs_host, torch.Tensor) else torch.from_numpy(
            np.ascontiguousarray(sun_dirs_host, dtype=np.float32))
        S = s.shape[0]
        if out_host is None:
            out_host = torch.empty((designs.D, S, 3), dtype=torch.float32)
        self._check(self.lib.srp_forces_host(self.handle, designs.handle, s.data_ptr(), S, rays_per_dir,
                                             max_bounces, seed, out_host.data_ptr()))
        return out_host

    def srp_first_hits(self, designs, sun_dirs, pairs, rays_per_dir, seed=0, method=0):
        pairs = self._pairs(designs, sun_dirs, pairs)
        out = torch.empty((pairs.shape[0], rays_per_dir), dtype=torch.int32, device=self.device)
        self._check(self.lib.srp_first_hits(self.handle, designs.handle, sun_dirs.data_ptr(), sun_dirs.shape[0],
                                            pairs.data_ptr(), pairs.shape[0], rays_per_dir, seed, method,
                                            out.data_ptr()))
        self.stream.synchronize()
        return out

    def srp_path_signatures(self, designs, sun_dirs, pairs, rays_per_dir, max_bounces, seed=0):
        pairs = self._pairs(designs, sun_dirs, pairs)
        out = torch.empty((pairs.shape[0], rays_per_dir), dtype=torch.int64, device=self.device)
        self._check(self.lib.srp_path_signatures(self.handle, designs.handle, sun_dirs.data_ptr(), sun_dirs.shape[0],
                                                 pairs.data_ptr(), pairs.shape[0], rays_per_dir, max_bounces, seed,
                                                 out.data_ptr()))
        self.stream.synchronize()
        return out

    def srp_get_stats(self):
        st = srp_stats()
        self._check(self.lib.srp_get_stats(self.handle, ctypes.byref(st)))
        return st.as_dict()

    def srp_probe_peaks(self):
        a, b = ctypes.c_double(), ctypes.c_double()
        self._check(self.lib.srp_probe_peaks(self.handle, ctypes.byref(a), ctypes.byref(b)))
        return {"fp32_tflops": a.value, "l2_read_gbs": b.value}
