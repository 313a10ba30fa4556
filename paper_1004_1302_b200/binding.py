"""Thin ctypes binding of include/splotch.h (argument marshalling only).

Every step of the render path runs in the CUDA library; PyTorch is used for device memory and
streams.  There is no CPU fallback: if libsplotch_b200.so is missing or cannot be loaded,
importing the symbols raises, and every compute call needs a CUDA device.

Functions carry the names of the C entry points.  Device arrays are torch CUDA tensors (or raw
integer device pointers); host arrays are numpy arrays or pinned torch CPU tensors.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libsplotch_b200.so")

SPLOTCH_MAX_TYPES = 4
SPLOTCH_OK = 0
SPLOTCH_ERR_INVALID_ARG = -1
SPLOTCH_ERR_WORKSPACE = -2
SPLOTCH_ERR_CUDA = -3
SPLOTCH_ERR_LIMIT = -4
SPLOTCH_ADDITIVE = 0
SPLOTCH_ABSORB = 1
SPLOTCH_RAW_SUM = 1
SPLOTCH_NO_TENSOR = 2
SPLOTCH_FORCE_TENSOR = 4

# every symbol include/splotch.h declares (checked by tests/test_abi.py against the header text)
EXPORTS = [
    "splotch_workspace_bytes", "splotch_render", "splotch_render_batch", "splotch_workspace_status", "splotch_count_pairs",
    "splotch_normalize", "splotch_field_range", "splotch_field_normalize", "splotch_tonemap_rgb8", "splotch_workspace_bytes_host", "splotch_render_host", "splotch_render_host_async", "splotch_debug_project",
    "splotch_debug_bins", "splotch_debug_workspace_bytes", "splotch_debug_stats", "splotch_debug_tensor_stats", "splotch_debug_scan",
    "splotch_scan_static",
    "splotch_sort_scratch_bytes", "splotch_debug_sort_pairs", "splotch_status_string",
    "splotch_last_cuda_error", "splotch_version", "splotch_profile_enable", "splotch_profile_read",
    "splotch_launch_count",
]


class SplotchError(RuntimeError):
    def __init__(self, fn: str, status: int):
        lib = _lib()
        msg = lib.splotch_status_string(status).decode()
        extra = f" (cudaError {lib.splotch_last_cuda_error()})" if status == SPLOTCH_ERR_CUDA else ""
        super().__init__(f"{fn}: {msg}{extra}")
        self.status = status


class splotch_particles(C.Structure):
    _fields_ = [("x", C.c_void_p), ("y", C.c_void_p), ("z", C.c_void_p), ("r", C.c_void_p), ("I", C.c_void_p),
                ("colval", C.c_void_p), ("type", C.c_void_p), ("vr", C.c_void_p), ("vg", C.c_void_p), ("vb", C.c_void_p)]


class splotch_camera(C.Structure):
    _fields_ = [("eye", C.c_float * 3), ("lookat", C.c_float * 3), ("up", C.c_float * 3), ("fov_deg", C.c_float),
                ("width", C.c_int32), ("height", C.c_int32)]


class splotch_colormap(C.Structure):
    _fields_ = [("emission", C.c_void_p), ("absorption", C.c_void_p), ("n_entries", C.c_int32), ("n_types", C.c_int32)]


class splotch_params(C.Structure):
    _fields_ = [("brightness", C.c_float * 4), ("abs_brightness", C.c_float * 4), ("mode", C.c_int32),
                ("support_f", C.c_float), ("z_near", C.c_float), ("flags", C.c_uint32)]


_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1004_1302_b200.build` "
                "(the render path has no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.splotch_status_string.restype = C.c_char_p
        lib.splotch_sort_scratch_bytes.restype = C.c_uint64
        lib.splotch_sort_scratch_bytes.argtypes = [C.c_int64]
        lib.splotch_launch_count.restype = C.c_ulonglong
        _LIB = lib
    return _LIB


def library_path() -> str:
    _lib()
    return LIB_PATH


def _ptr(t) -> Optional[int]:
    """Device or host address of a tensor / array / int; None stays NULL."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return int(t.data_ptr())
    if hasattr(t, "ctypes"):
        return int(t.ctypes.data)
    raise TypeError(f"cannot take the address of {type(t)}")


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)


def make_particles(x, y, z, r, I, colval, type=None, vec=None) -> splotch_particles:
    """vec: optional (vr, vg, vb) arrays for vector colouring (colval may then be None)."""
    v = (None, None, None) if vec is None else vec
    return splotch_particles(_ptr(x), _ptr(y), _ptr(z), _ptr(r), _ptr(I), _ptr(colval), _ptr(type),
                             _ptr(v[0]), _ptr(v[1]), _ptr(v[2]))


def make_camera(eye: Sequence[float], lookat: Sequence[float], up: Sequence[float], fov_deg: float, width: int,
                height: int) -> splotch_camera:
    f3 = C.c_float * 3
    return splotch_camera(f3(*eye), f3(*lookat), f3(*up), float(fov_deg), int(width), int(height))


def make_colormap(emission, absorption, n_entries: int, n_types: int) -> splotch_colormap:
    return splotch_colormap(_ptr(emission), _ptr(absorption), int(n_entries), int(n_types))


def make_params(brightness: Sequence[float], abs_brightness: Optional[Sequence[float]] = None, mode: int = 0,
                support_f: float = 3.0, z_near: float = 0.01, flags: int = 0) -> splotch_params:
    b = list(brightness) + [0.0] * (4 - len(brightness))
    a = list(abs_brightness if abs_brightness is not None else brightness)
    a = a + [0.0] * (4 - len(a))
    f4 = C.c_float * 4
    return splotch_params(f4(*b[:4]), f4(*a[:4]), int(mode), float(support_f), float(z_near), int(flags))


def _check(fn: str, status: int) -> None:
    if status != SPLOTCH_OK:
        raise SplotchError(fn, status)


def _vp(v):
    return C.c_void_p(v)


# --------------------------------------------------------------------------------------------
# entry points (same names and argument order as the header)
# --------------------------------------------------------------------------------------------
def splotch_version() -> int:
    return int(_lib().splotch_version())


def splotch_status_string(status: int) -> str:
    return _lib().splotch_status_string(int(status)).decode()


def splotch_last_cuda_error() -> int:
    return int(_lib().splotch_last_cuda_error())


def splotch_workspace_bytes(n: int, camera: splotch_camera, params: splotch_params, max_pairs: int) -> int:
    out = C.c_uint64(0)
    _check("splotch_workspace_bytes", _lib().splotch_workspace_bytes(C.c_int64(n), C.byref(camera), C.byref(params),
                                                                    C.c_uint64(max_pairs), C.byref(out)))
    return int(out.value)


def splotch_workspace_bytes_host(n: int, camera: splotch_camera, colormap_host: splotch_colormap,
                                 params: splotch_params, max_pairs: int) -> int:
    out = C.c_uint64(0)
    _check("splotch_workspace_bytes_host",
           _lib().splotch_workspace_bytes_host(C.c_int64(n), C.byref(camera), C.byref(colormap_host), C.byref(params),
                                               C.c_uint64(max_pairs), C.byref(out)))
    return int(out.value)


def splotch_debug_workspace_bytes(n: int, camera: splotch_camera, params: splotch_params, bin_shift: int,
                                  max_members: int) -> int:
    out = C.c_uint64(0)
    _check("splotch_debug_workspace_bytes",
           _lib().splotch_debug_workspace_bytes(C.c_int64(n), C.byref(camera), C.byref(params), C.c_int32(bin_shift),
                                                C.c_uint64(max_members), C.byref(out)))
    return int(out.value)


def splotch_render(particles: splotch_particles, n: int, camera: splotch_camera, colormap: splotch_colormap,
                   params: splotch_params, out_rgb, workspace, workspace_bytes: int, max_pairs: int, stream=None) -> None:
    _check("splotch_render",
           _lib().splotch_render(C.byref(particles), C.c_int64(n), C.byref(camera), C.byref(colormap), C.byref(params),
                                 _vp(_ptr(out_rgb)), _vp(_ptr(workspace)), C.c_uint64(workspace_bytes),
                                 C.c_uint64(max_pairs), _vp(_stream(stream))))


def splotch_render_batch(particles: splotch_particles, n: int, cameras: Sequence[splotch_camera], colormap: splotch_colormap,
                         params: splotch_params, out_rgb, frame_status, workspace, workspace_bytes: int, max_pairs: int,
                         stream=None) -> None:
    """K cameras over one resident particle set: out_rgb holds K images back to back, frame_status (device, K*4 uint64
    as int64 tensor, or None) receives per frame (status, visible, pairs, 0).  Enqueue only."""
    arr = (splotch_camera * max(len(cameras), 1))(*cameras)
    _check("splotch_render_batch",
           _lib().splotch_render_batch(C.byref(particles), C.c_int64(n), arr, C.c_int32(len(cameras)), C.byref(colormap),
                                       C.byref(params), _vp(_ptr(out_rgb)), _vp(_ptr(frame_status)), _vp(_ptr(workspace)),
                                       C.c_uint64(workspace_bytes), C.c_uint64(max_pairs), _vp(_stream(stream))))


def splotch_workspace_status(workspace, stream=None):
    """(status, visible, pairs); synchronises the stream."""
    st, vis, pairs = C.c_int32(0), C.c_uint64(0), C.c_uint64(0)
    _check("splotch_workspace_status",
           _lib().splotch_workspace_status(_vp(_ptr(workspace)), _vp(_stream(stream)), C.byref(st), C.byref(vis),
                                           C.byref(pairs)))
    return int(st.value), int(vis.value), int(pairs.value)


def splotch_count_pairs(particles: splotch_particles, n: int, camera: splotch_camera, colormap: splotch_colormap,
                        params: splotch_params, workspace, workspace_bytes: int, stream=None):
    """(pairs, visible); synchronises the stream."""
    pairs, vis = C.c_uint64(0), C.c_uint64(0)
    _check("splotch_count_pairs",
           _lib().splotch_count_pairs(C.byref(particles), C.c_int64(n), C.byref(camera), C.byref(colormap),
                                      C.byref(params), _vp(_ptr(workspace)), C.c_uint64(workspace_bytes),
                                      C.byref(pairs), C.byref(vis), _vp(_stream(stream))))
    return int(pairs.value), int(vis.value)


def splotch_normalize(S, out, n_values: int, stream=None) -> None:
    _check("splotch_normalize", _lib().splotch_normalize(_vp(_ptr(S)), _vp(_ptr(out)), C.c_int64(n_values),
                                                         _vp(_stream(stream))))


def splotch_field_range(values, n: int, log_scale: bool, range_out, stream=None) -> None:
    _check("splotch_field_range", _lib().splotch_field_range(_vp(_ptr(values)), C.c_int64(n), C.c_int32(1 if log_scale else 0),
                                                           _vp(_ptr(range_out)), _vp(_stream(stream))))


def splotch_field_normalize(values, n: int, log_scale: bool, range_in, out, stream=None) -> None:
    _check("splotch_field_normalize",
           _lib().splotch_field_normalize(_vp(_ptr(values)), C.c_int64(n), C.c_int32(1 if log_scale else 0),
                                          _vp(_ptr(range_in)), _vp(_ptr(out)), _vp(_stream(stream))))


def splotch_tonemap_rgb8(rgb, n_values: int, gamma: float, out, stream=None) -> None:
    _check("splotch_tonemap_rgb8", _lib().splotch_tonemap_rgb8(_vp(_ptr(rgb)), C.c_int64(n_values), C.c_float(gamma),
                                                             _vp(_ptr(out)), _vp(_stream(stream))))


def splotch_render_host(particles_host: splotch_particles, n: int, camera: splotch_camera,
                        colormap_host: splotch_colormap, params: splotch_params, out_rgb_host, workspace,
                        workspace_bytes: int, max_pairs: int, stream=None) -> None:
    _check("splotch_render_host",
           _lib().splotch_render_host(C.byref(particles_host), C.c_int64(n), C.byref(camera), C.byref(colormap_host),
                                      C.byref(params), _vp(_ptr(out_rgb_host)), _vp(_ptr(workspace)),
                                      C.c_uint64(workspace_bytes), C.c_uint64(max_pairs), _vp(_stream(stream))))


def splotch_render_host_async(particles_host: splotch_particles, n: int, camera: splotch_camera,
                              colormap_host: splotch_colormap, params: splotch_params, out_rgb_host, workspace,
                              workspace_bytes: int, max_pairs: int, stream=None) -> None:
    """Enqueue only: H2D copies, render, D2H copy of the image on `stream`; check later with splotch_workspace_status."""
    _check("splotch_render_host_async",
           _lib().splotch_render_host_async(C.byref(particles_host), C.c_int64(n), C.byref(camera), C.byref(colormap_host),
                                            C.byref(params), _vp(_ptr(out_rgb_host)), _vp(_ptr(workspace)),
                                            C.c_uint64(workspace_bytes), C.c_uint64(max_pairs), _vp(_stream(stream))))


def splotch_debug_project(particles, n, camera, colormap, params, workspace, workspace_bytes, sx, sy, sigma_s, R, zkey,
                          pix_bbox, visible, stream=None) -> None:
    _check("splotch_debug_project",
           _lib().splotch_debug_project(C.byref(particles), C.c_int64(n), C.byref(camera), C.byref(colormap),
                                        C.byref(params), _vp(_ptr(workspace)), C.c_uint64(workspace_bytes),
                                        _vp(_ptr(sx)), _vp(_ptr(sy)), _vp(_ptr(sigma_s)), _vp(_ptr(R)), _vp(_ptr(zkey)),
                                        _vp(_ptr(pix_bbox)), _vp(_ptr(visible)), _vp(_stream(stream))))


def splotch_debug_bins(particles, n, camera, colormap, params, workspace, workspace_bytes, bin_shift, tile_count,
                       tile_offset, member_ids, max_members, stream=None) -> None:
    _check("splotch_debug_bins",
           _lib().splotch_debug_bins(C.byref(particles), C.c_int64(n), C.byref(camera), C.byref(colormap),
                                     C.byref(params), _vp(_ptr(workspace)), C.c_uint64(workspace_bytes),
                                     C.c_int32(bin_shift), _vp(_ptr(tile_count)), _vp(_ptr(tile_offset)),
                                     _vp(_ptr(member_ids)), C.c_uint64(max_members), _vp(_stream(stream))))


def splotch_debug_stats(particles, n, camera, colormap, params, workspace, workspace_bytes, bin_shift, stream=None):
    """(visible, pairs, updates); synchronises the stream."""
    vis, pairs, upd = C.c_uint64(0), C.c_uint64(0), C.c_uint64(0)
    _check("splotch_debug_stats",
           _lib().splotch_debug_stats(C.byref(particles), C.c_int64(n), C.byref(camera), C.byref(colormap),
                                      C.byref(params), _vp(_ptr(workspace)), C.c_uint64(workspace_bytes),
                                      C.c_int32(bin_shift), C.byref(vis), C.byref(pairs), C.byref(upd),
                                      _vp(_stream(stream))))
    return int(vis.value), int(pairs.value), int(upd.value)


def splotch_debug_tensor_stats(particles, n, camera, colormap, params, workspace, workspace_bytes, stream=None):
    """(updates on the tensor cores, tensor_on chosen by the library, estimated share); synchronises the stream."""
    upd, on, share = C.c_uint64(0), C.c_int32(0), C.c_float(0.0)
    _check("splotch_debug_tensor_stats",
           _lib().splotch_debug_tensor_stats(C.byref(particles), C.c_int64(n), C.byref(camera), C.byref(colormap),
                                             C.byref(params), _vp(_ptr(workspace)), C.c_uint64(workspace_bytes),
                                             C.byref(upd), C.byref(on), C.byref(share), _vp(_stream(stream))))
    return int(upd.value), int(on.value), float(share.value)


def splotch_debug_scan(inp, out, n: int, scratch, scratch_bytes: int, stream=None) -> None:
    _check("splotch_debug_scan", _lib().splotch_debug_scan(_vp(_ptr(inp)), _vp(_ptr(out)), C.c_int64(n),
                                                           _vp(_ptr(scratch)), C.c_uint64(scratch_bytes),
                                                           _vp(_stream(stream))))


SPLOTCH_SCAN_STATIC_MAX_N = 1 << 24


def splotch_scan_static(inp, out, n: int, stream=None) -> None:
    """Exclusive scan of n uint32 counts into n + 1 uint64 offsets, like splotch_debug_scan, for callers that cannot
    give the library scratch memory and are not allowed to allocate any (a renderer embedded in a simulation whose own
    pool holds all of the GPU's memory): the scan's bookkeeping sits in a fixed 66,048-byte array inside the library.
    n <= SPLOTCH_SCAN_STATIC_MAX_N, else SplotchError(SPLOTCH_ERR_LIMIT).  Calls on one device share that array: keep
    them on one stream or order them.  Marshalling only; see include/splotch.h."""
    _check("splotch_scan_static", _lib().splotch_scan_static(_vp(_ptr(inp)), _vp(_ptr(out)), C.c_int64(n),
                                                             _vp(_stream(stream))))


def splotch_sort_scratch_bytes(n: int) -> int:
    return int(_lib().splotch_sort_scratch_bytes(C.c_int64(n)))


def splotch_debug_sort_pairs(keys, vals, keys_tmp, vals_tmp, n: int, key_bits: int, scratch, scratch_bytes: int,
                             stream=None) -> None:
    _check("splotch_debug_sort_pairs",
           _lib().splotch_debug_sort_pairs(_vp(_ptr(keys)), _vp(_ptr(vals)), _vp(_ptr(keys_tmp)), _vp(_ptr(vals_tmp)),
                                           C.c_int64(n), C.c_int32(key_bits), _vp(_ptr(scratch)),
                                           C.c_uint64(scratch_bytes), _vp(_stream(stream))))


def splotch_profile_enable(on: bool) -> None:
    _check("splotch_profile_enable", _lib().splotch_profile_enable(C.c_int(1 if on else 0)))


def splotch_profile_read():
    """(list of 6 mean stage times in ms, number of profiled calls); synchronises."""
    ms = (C.c_double * 6)()
    calls = C.c_int64(0)
    _check("splotch_profile_read", _lib().splotch_profile_read(ms, C.byref(calls)))
    return [float(v) for v in ms], int(calls.value)


def splotch_launch_count() -> int:
    return int(_lib().splotch_launch_count())
