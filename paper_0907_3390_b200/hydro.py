"""Thin Python binding of include/gamer_hydro.h (ctypes; argument marshalling only).

Every function here has the name of the C entry point it calls.  Device buffers are torch CUDA tensors (or raw
integer device pointers); nothing is computed in Python.  If libgamer_hydro.so is missing or fails to load this
module raises — there is no fallback of any kind.
"""
import ctypes
import os

GAMER_OK, GAMER_EINVAL, GAMER_EUNSUPPORTED, GAMER_ECUDA, GAMER_ENOMEM = 0, -1, -2, -3, -4
NCOMP, PS, NGHOST, NP = 5, 16, 3, 22
IN_GROUP_FLOATS = NCOMP * NP ** 3
OUT_GROUP_FLOATS = NCOMP * PS ** 3
FACE_GROUP_FLOATS = 3 * 3 * NCOMP * PS * PS

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgamer_hydro.so")
_lib = None


class GamerError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("gamer_hydro: status %d: %s" % (code, msg))
        self.code = code


def lib():
    """Load libgamer_hydro.so (built by `python -m paper_0907_3390_b200.build`).  Fails loudly if it is absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not found: build it with `python -m paper_0907_3390_b200.build` "
                              "(there is no CPU fallback)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        L.gamer_hydro_abi_version.restype = ctypes.c_int
        if L.gamer_hydro_abi_version() != ABI_VERSION:
            raise ImportError("%s has ABI version %d, this binding needs %d: rebuild it"
                              % (LIB_PATH, L.gamer_hydro_abi_version(), ABI_VERSION))
        vp, ll, ci, cf = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int, ctypes.c_float
        L.gamer_hydro_advance.restype = ci
        L.gamer_hydro_advance.argtypes = [vp, vp, ll, ci, cf, cf, cf, vp]
        L.gamer_hydro_advance_ex.restype = ci
        L.gamer_hydro_advance_ex.argtypes = [vp, vp, ll, ci, cf, cf, cf, ci, vp, vp, vp]
        L.gamer_hydro_in_floats.restype = ctypes.c_size_t
        L.gamer_hydro_in_floats.argtypes = [ll, ci]
        L.gamer_hydro_out_floats.restype = ctypes.c_size_t
        L.gamer_hydro_out_floats.argtypes = [ll]
        L.gamer_hydro_face_flux_floats.restype = ctypes.c_size_t
        L.gamer_hydro_face_flux_floats.argtypes = [ll]
        L.gamer_hydro_pipeline_run.restype = ci
        L.gamer_hydro_pipeline_run.argtypes = [vp, vp, ll, ci, cf, cf, cf, ci, ll, ci]
        L.gamer_hydro_pipeline_release.restype = ci
        L.gamer_hydro_pipeline_release.argtypes = []
        L.gamer_hydro_ghost_fill.restype = ci
        L.gamer_hydro_ghost_fill.argtypes = [vp, vp, ci, ci, ci, ci, ci, ci, vp]
        L.gamer_hydro_run_uniform.restype = ci
        L.gamer_hydro_run_uniform.argtypes = [vp, vp, ci, ci, ci, ci, ci, ci, ci, ci, cf, cf, cf, vp, vp, vp]
        L.gamer_hydro_run_uniform_noalloc.restype = ci
        L.gamer_hydro_run_uniform_noalloc.argtypes = [vp, vp, ci, ci, ci, ci, ci, ci, ci, ci, cf, cf, cf, vp, vp]
        L.gamer_hydro_noalloc_max_groups.restype = ll
        L.gamer_hydro_noalloc_max_groups.argtypes = []
        L.gamer_hydro_advance_f64_ex.restype = ci
        L.gamer_hydro_advance_f64_ex.argtypes = [vp, vp, ll, ci, ctypes.c_double, ctypes.c_double, ctypes.c_double, ci, vp, vp, vp]
        L.gamer_hydro_launch_info.restype = ci
        L.gamer_hydro_launch_info.argtypes = [ll] + [ctypes.POINTER(ci)] * 4
        L.gamer_last_error.restype = ctypes.c_char_p
        L.gamer_last_error.argtypes = []
        L.gamer_version.restype = ctypes.c_char_p
        L.gamer_version.argtypes = []
        L.gamer_hydro_abi_version.restype = ci
        L.gamer_hydro_abi_version.argtypes = []
        _lib = L
    return _lib


def _ptr(x):
    """Raw address of a torch tensor / numpy array / int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError("cannot take the address of %r" % type(x))


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _check(rc):
    if rc != GAMER_OK:
        raise GamerError(rc, gamer_last_error())


def gamer_last_error():
    return lib().gamer_last_error().decode()


def gamer_version():
    return lib().gamer_version().decode()


ABI_VERSION = 3          # GAMER_HYDRO_ABI_VERSION of the header this binding was written against


def gamer_hydro_abi_version():
    return int(lib().gamer_hydro_abi_version())


def gamer_hydro_in_floats(n_groups, ghost=NGHOST):
    return int(lib().gamer_hydro_in_floats(n_groups, ghost))


def gamer_hydro_out_floats(n_groups):
    return int(lib().gamer_hydro_out_floats(n_groups))


def gamer_hydro_face_flux_floats(n_groups):
    return int(lib().gamer_hydro_face_flux_floats(n_groups))


def gamer_hydro_advance(d_in, d_out, n_groups, ghost, dt, dh, gamma, stream=None, check=True):
    """Enqueue one forward (x,y,z) pass on `stream` (default: torch's current stream).  Returns the status code."""
    rc = lib().gamer_hydro_advance(_ptr(d_in), _ptr(d_out), n_groups, ghost, dt, dh, gamma, _stream_ptr(stream))
    if check:
        _check(rc)
    return rc


def gamer_hydro_advance_ex(d_in, d_out, n_groups, ghost, dt, dh, gamma, backward=0, d_face_flux=None,
                           d_group_maxspeed=None, stream=None, check=True):
    rc = lib().gamer_hydro_advance_ex(_ptr(d_in), _ptr(d_out), n_groups, ghost, dt, dh, gamma, int(backward),
                                      _ptr(d_face_flux), _ptr(d_group_maxspeed), _stream_ptr(stream))
    if check:
        _check(rc)
    return rc


def gamer_hydro_pipeline_run(h_in, h_out, n_groups, ghost, dt, dh, gamma, backward=0, groups_per_chunk=1024,
                             n_streams=4, check=True):
    """Host buffers in, host buffers out (pinned for overlap), synchronous (Fig.5)."""
    rc = lib().gamer_hydro_pipeline_run(_ptr(h_in), _ptr(h_out), n_groups, ghost, dt, dh, gamma, int(backward),
                                        groups_per_chunk, n_streams)
    if check:
        _check(rc)
    return rc


def gamer_hydro_pipeline_release(check=True):
    """Free the streams and staging buffers that gamer_hydro_pipeline_run keeps between calls."""
    rc = lib().gamer_hydro_pipeline_release()
    if check:
        _check(rc)
    return rc


def gamer_hydro_ghost_fill(d_interior, d_padded, gx, gy, gz, bc_x=0, bc_y=0, bc_z=0, stream=None, check=True):
    """Device-side ghost fill of a single-level tiling of gx*gy*gz groups.  bc: 0 periodic, 1 keep."""
    rc = lib().gamer_hydro_ghost_fill(_ptr(d_interior), _ptr(d_padded), gx, gy, gz, bc_x, bc_y, bc_z,
                                      _stream_ptr(stream))
    if check:
        _check(rc)
    return rc


def gamer_hydro_run_uniform(d_padded, d_interior, gx, gy, gz, bc_x, bc_y, bc_z, n_steps, order, cfl, dh, gamma, d_work,
                            d_dt_log=None, stream=None, check=True):
    """n_steps of {CFL dt on the device, forward pass, ghost fill [, backward pass with the same dt, ghost fill if
    order = 1]} without leaving the device."""
    rc = lib().gamer_hydro_run_uniform(_ptr(d_padded), _ptr(d_interior), gx, gy, gz, bc_x, bc_y, bc_z, n_steps,
                                       int(order), cfl, dh, gamma, _ptr(d_work), _ptr(d_dt_log), _stream_ptr(stream))
    if check:
        _check(rc)
    return rc


def gamer_hydro_run_uniform_noalloc(d_padded, d_interior, gx, gy, gz, bc_x, bc_y, bc_z, n_steps, order, cfl, dh, gamma,
                                    d_dt_log=None, stream=None, check=True):
    """gamer_hydro_run_uniform without d_work, for callers that cannot allocate device memory (their pool owns it
    all, or an allocation would stall the other streams of a running time-step loop): the scratch is a fixed array
    inside the library, good for boxes of up to gamer_hydro_noalloc_max_groups() groups (larger ones are refused).
    One array per GPU, shared by all calls: do not let two of them overlap on the same GPU.  Make the first call on a
    device during start-up (n_steps = 0 does nothing else) and before any stream capture."""
    rc = lib().gamer_hydro_run_uniform_noalloc(_ptr(d_padded), _ptr(d_interior), gx, gy, gz, bc_x, bc_y, bc_z, n_steps,
                                               int(order), cfl, dh, gamma, _ptr(d_dt_log), _stream_ptr(stream))
    if check:
        _check(rc)
    return rc


def gamer_hydro_noalloc_max_groups():
    return int(lib().gamer_hydro_noalloc_max_groups())


def gamer_hydro_advance_f64_ex(d_in, d_out, n_groups, ghost, dt, dh, gamma, backward=0, d_face_flux=None,
                               d_group_maxspeed=None, stream=None, check=True):
    """One pass in double precision with the optional outputs (face fluxes, per-group CFL speed) in double."""
    rc = lib().gamer_hydro_advance_f64_ex(_ptr(d_in), _ptr(d_out), n_groups, ghost, dt, dh, gamma, int(backward),
                                          _ptr(d_face_flux), _ptr(d_group_maxspeed), _stream_ptr(stream))
    if check:
        _check(rc)
    return rc


def gamer_hydro_launch_info(n_groups):
    g, b, s, r = (ctypes.c_int(0) for _ in range(4))
    _check(lib().gamer_hydro_launch_info(n_groups, ctypes.byref(g), ctypes.byref(b), ctypes.byref(s), ctypes.byref(r)))
    return dict(grid=g.value, block=b.value, smem_bytes=s.value, regs_per_thread=r.value)
