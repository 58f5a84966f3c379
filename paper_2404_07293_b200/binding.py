"""Thin ctypes binding over libscw.so (include/scwatter.h): argument marshalling only.

PyTorch supplies device memory and the CUDA stream; every step of the path runs in the
library's kernels.  There is no CPU fallback: importing is cheap, but any call raises
ScwError / RuntimeError if libscw.so is missing or the device is not an sm_100 GPU.
"""
import ctypes
import os
from ctypes import (POINTER, Structure, byref, c_char_p, c_double, c_int8, c_int32, c_int64, c_size_t,
                    c_uint32, c_void_p)

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libscw.so")

SCW_C64, SCW_C128 = 0, 1
SCW_MODES_PLANEWAVE, SCW_MODES_DENSE = 0, 1
SCW_OPT_PATH, SCW_OPT_PROFILE, SCW_OPT_CACHE = 1, 2, 3
SCW_PATH_AUTO, SCW_PATH_SIMT, SCW_PATH_TENSOR = 0, 1, 2
STATUS = {0: "SCW_OK", 1: "SCW_ERR_NULL", 2: "SCW_ERR_SHAPE", 3: "SCW_ERR_DTYPE", 4: "SCW_ERR_ALIGN",
          5: "SCW_ERR_VALUE", 6: "SCW_ERR_WORKSPACE", 7: "SCW_ERR_CUDA", 8: "SCW_ERR_UNSUPPORTED"}

EXPORTS = [
    "scw_version", "scw_create", "scw_destroy", "scw_set_stream", "scw_set_workspace", "scw_set_option",
    "scw_last_error", "scw_last_cuda_error", "scw_required_workspace", "scw_launch_count", "scw_last_kernels",
    "scw_assemble_spectra", "scw_assemble_workspace", "scw_synthesize_grid", "scw_synthesize_workspace",
    "scw_eval_points", "scw_points_workspace", "scw_eval_points_noalloc", "scw_sweep_wavelengths", "scw_sweep_workspace",
    "scw_sweep_wavelengths_host", "scw_sweep_host_workspace",
    "scw_profile_classes", "scw_profile_name", "scw_profile_read", "scw_profile_reset",
    "scw_exterior_spectra", "scw_exterior_points", "scw_exterior_points_workspace", "scw_exterior_grid",
    "scw_exterior_grid_workspace",
    "scw_sweep_intensity", "scw_sweep_intensity_workspace",
    "scw_measure_peak", "scw_invalidate_cache", "scw_calibrate", "scw_profile_assembly", "scw_profile_timeline",
    "scw_sweep_detector", "scw_sweep_detector_workspace", "scw_absorbance", "scw_build_V", "scw_build_V_workspace", "scw_propagate_alpha", "scw_propagate_alpha_workspace",
]
SCW_PEAKS = {"fp64_dmma_tflops": 0, "fp32_fma_tflops": 1, "mufu_gops": 2, "hbm_read_gbs": 3, "hbm_write_gbs": 4,
             "hbm_write_tma_gbs": 5, "mufu_sincosex2_gops": 6}
SCW_SIDE_ABOVE, SCW_SIDE_BELOW = 0, 1


class scw_exterior(Structure):
    _fields_ = [("struct_size", c_uint32), ("dtype", c_int32), ("side", c_int32), ("U", c_int32), ("Vn", c_int32),
                ("X", c_double), ("Y", c_double), ("lambda_", c_double), ("n_re", c_double), ("n_im", c_double),
                ("z_face", c_double), ("z_inc", c_double), ("p_face", c_void_p), ("p_inc", c_void_p)]


class scw_vbuild(Structure):
    _fields_ = [("struct_size", c_uint32), ("dtype", c_int32), ("U", c_int32), ("Vn", c_int32), ("X", c_double),
                ("Y", c_double), ("lambda_", c_double), ("J", c_int64), ("Q", c_void_p), ("ldQ", c_int64), ("psi", c_void_p),
                ("alpha", c_void_p)]


class scw_stack(Structure):
    _fields_ = [("struct_size", c_uint32), ("dtype", c_int32), ("n_layers", c_int32), ("n", c_int64), ("lambda_", c_double),
                ("z_if", POINTER(c_double)), ("Q", POINTER(c_void_p)), ("ldQ", c_int64), ("gamma", POINTER(c_void_p)),
                ("dir", POINTER(c_void_p))]


class scw_window(Structure):
    _fields_ = [("ix0", c_int64), ("ix1", c_int64), ("iy0", c_int64), ("iy1", c_int64)]


class ScwError(RuntimeError):
    def __init__(self, status, message=""):
        self.status = status
        super().__init__(f"{STATUS.get(status, status)}: {message}")


class scw_layer(Structure):
    _fields_ = [("struct_size", c_uint32), ("dtype", c_int32), ("U", c_int32), ("Vn", c_int32),
                ("X", c_double), ("Y", c_double), ("lambda_", c_double), ("z_lo", c_double), ("z_hi", c_double),
                ("J", c_int64), ("V", c_void_p), ("ldV", c_int64), ("c", c_void_p), ("gamma", c_void_p),
                ("dir", c_void_p)]


class scw_modes(Structure):
    _fields_ = [("struct_size", c_uint32), ("kind", c_int32), ("dtype", c_int32), ("J", c_int64),
                ("lambda_", c_double), ("sx", c_void_p), ("sy", c_void_p), ("gamma", c_void_p),
                ("zref", c_void_p), ("p", c_void_p), ("layer", scw_layer)]


_LIB = None


def lib():
    """Load libscw.so (built in-tree by paper_2404_07293_b200.build); fail loudly if absent."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2404_07293_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        L.scw_last_error.restype = c_char_p
        L.scw_required_workspace.restype = c_size_t
        L.scw_launch_count.restype = c_int64
        L.scw_create.argtypes = [POINTER(c_void_p), c_int32, c_void_p]
        L.scw_destroy.argtypes = [c_void_p]
        L.scw_set_stream.argtypes = [c_void_p, c_void_p]
        L.scw_set_workspace.argtypes = [c_void_p, c_void_p, c_size_t]
        L.scw_set_option.argtypes = [c_void_p, c_int32, c_int64]
        L.scw_last_error.argtypes = [c_void_p]
        L.scw_last_cuda_error.argtypes = [c_void_p]
        L.scw_required_workspace.argtypes = [c_void_p]
        L.scw_launch_count.argtypes = [c_void_p]
        L.scw_last_kernels.restype = ctypes.c_uint64
        L.scw_last_kernels.argtypes = [c_void_p]
        L.scw_profile_name.restype = c_char_p
        L.scw_profile_name.argtypes = [c_int32]
        L.scw_profile_read.argtypes = [c_void_p, c_int32, POINTER(c_double), POINTER(c_int64)]
        L.scw_profile_reset.argtypes = [c_void_p]
        L.scw_assemble_spectra.argtypes = [c_void_p, POINTER(scw_layer), c_int64, c_void_p, c_void_p, c_int64]
        L.scw_assemble_workspace.argtypes = [c_void_p, POINTER(scw_layer), c_int64, POINTER(c_size_t)]
        L.scw_synthesize_grid.argtypes = [c_void_p, c_int32, c_int32, c_int32, c_double, c_double, c_int64,
                                          c_void_p, c_int64, c_int64, c_void_p, c_int64, c_void_p, c_void_p,
                                          POINTER(c_int64)]
        L.scw_synthesize_workspace.argtypes = [c_void_p, c_int32, c_int32, c_int32, c_int64, c_int64, c_int64,
                                               POINTER(c_size_t)]
        L.scw_eval_points.argtypes = [c_void_p, POINTER(scw_modes), c_int64, c_void_p, c_void_p]
        L.scw_points_workspace.argtypes = [c_void_p, POINTER(scw_modes), c_int64, POINTER(c_size_t)]
        L.scw_eval_points_noalloc.argtypes = [c_void_p, POINTER(scw_modes), c_int64, c_void_p, c_void_p]
        L.scw_sweep_wavelengths.argtypes = [c_void_p, c_int64, POINTER(scw_layer), POINTER(c_int64),
                                            POINTER(c_void_p), c_int64, c_void_p, c_int64, c_void_p,
                                            POINTER(c_void_p), POINTER(c_int64)]
        L.scw_sweep_workspace.argtypes = [c_void_p, c_int64, POINTER(scw_layer), POINTER(c_int64), c_int64,
                                          c_int64, POINTER(c_size_t)]
        L.scw_sweep_wavelengths_host.argtypes = [c_void_p, c_int64, POINTER(scw_layer), POINTER(c_int64),
                                                 POINTER(c_void_p), c_int64, c_void_p, c_int64, c_void_p,
                                                 POINTER(c_void_p), POINTER(c_int64), POINTER(c_int64)]
        L.scw_sweep_host_workspace.argtypes = [c_void_p, c_int64, POINTER(scw_layer), POINTER(c_int64), c_int64,
                                               c_int64, POINTER(c_size_t)]
        L.scw_sweep_intensity.argtypes = L.scw_sweep_wavelengths.argtypes
        L.scw_sweep_intensity_workspace.argtypes = L.scw_sweep_workspace.argtypes
        L.scw_exterior_spectra.argtypes = [c_void_p, POINTER(scw_exterior), c_int64, c_void_p, c_void_p, c_int64]
        L.scw_exterior_grid.argtypes = [c_void_p, POINTER(scw_exterior), c_int64, c_void_p, c_int64, c_void_p, c_int64, c_void_p,
                                        c_void_p, POINTER(c_int64)]
        L.scw_exterior_grid_workspace.argtypes = [c_void_p, POINTER(scw_exterior), c_int64, c_int64, c_int64, POINTER(c_size_t)]
        L.scw_exterior_points.argtypes = [c_void_p, POINTER(scw_exterior), c_int64, c_void_p, c_void_p]
        L.scw_exterior_points_workspace.argtypes = [c_void_p, POINTER(scw_exterior), c_int64, POINTER(c_size_t)]
        L.scw_sweep_detector.argtypes = L.scw_sweep_wavelengths.argtypes + [POINTER(scw_window), POINTER(c_void_p)]
        L.scw_sweep_detector_workspace.argtypes = L.scw_sweep_workspace.argtypes
        L.scw_absorbance.argtypes = [c_void_p, c_int32, c_int64, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
        L.scw_build_V.argtypes = [c_void_p, POINTER(scw_vbuild), c_void_p, c_int64]
        L.scw_build_V_workspace.argtypes = [c_void_p, POINTER(scw_vbuild), POINTER(c_size_t)]
        L.scw_propagate_alpha.argtypes = [c_void_p, POINTER(scw_stack), c_void_p, POINTER(c_void_p), c_void_p]
        L.scw_propagate_alpha_workspace.argtypes = [c_void_p, POINTER(scw_stack), POINTER(c_size_t)]
        L.scw_invalidate_cache.argtypes = [c_void_p]
        L.scw_profile_assembly.argtypes = [c_void_p, c_int32, POINTER(c_double), POINTER(c_int32)]
        L.scw_profile_timeline.argtypes = [c_void_p, c_int32, POINTER(ctypes.c_uint64), POINTER(c_int32), POINTER(c_int32)]
        L.scw_calibrate.argtypes = L.scw_sweep_wavelengths.argtypes + [c_int32]
        L.scw_measure_peak.argtypes = [c_void_p, c_int32, c_void_p, c_size_t, c_int32, POINTER(c_double)]
        _LIB = L
    return _LIB


def _dt(t):
    if t.dtype == torch.complex64:
        return SCW_C64
    if t.dtype == torch.complex128:
        return SCW_C128
    raise ScwError(3, f"unsupported tensor dtype {t.dtype}")


def _p(t):
    return None if t is None else c_void_p(t.data_ptr())


class Layer:
    """Tensors of one layer at one wavelength (device tensors, or host tensors for the *_host call).

    V: (J, ldV) complex (column-major [ldV x J]); c: (J,) complex or None; gamma: (J,) complex128;
    dir: (J,) int8 or None.
    """

    def __init__(self, *, U, Vn, X, Y, lam, z_lo, z_hi, V, gamma, c=None, dir=None, **_):
        self.U, self.Vn, self.X, self.Y, self.lam = int(U), int(Vn), float(X), float(Y), float(lam)
        self.z_lo, self.z_hi = float(z_lo), float(z_hi)
        self.V, self.c, self.gamma, self.dir = V, c, gamma, dir
        self._struct = None
        assert V.dim() == 2 and V.is_contiguous() and gamma.dtype == torch.complex128
        assert c is None or c.dtype == V.dtype
        assert dir is None or dir.dtype == torch.int8

    @property
    def J(self):
        return self.V.shape[0]

    @property
    def R(self):
        return 3 * self.U * self.Vn

    def struct(self):
        """A fresh scw_layer descriptor of this layer (the caller may edit it)."""
        return scw_layer(ctypes.sizeof(scw_layer), _dt(self.V), self.U, self.Vn, self.X, self.Y, self.lam,
                         self.z_lo, self.z_hi, self.V.shape[0], self.V.data_ptr(), self.V.shape[1],
                         None if self.c is None else self.c.data_ptr(), self.gamma.data_ptr(),
                         None if self.dir is None else self.dir.data_ptr())

    def _cached_struct(self):
        """The descriptor built once, for the sweep calls that marshal many layers per call (a Layer is not modified after
        construction; never handed out)."""
        if self._struct is None:
            self._struct = self.struct()
        return self._struct

    @staticmethod
    def from_numpy(d, device):
        """Upload a scw_inputs / oracle-style dict of numpy arrays."""
        t = lambda a: None if a is None else torch.from_numpy(a).to(device)
        return Layer(U=d["U"], Vn=d["Vn"], X=d["X"], Y=d["Y"], lam=d["lam"], z_lo=d["z_lo"], z_hi=d["z_hi"],
                     V=t(d["V"]), gamma=t(d["gamma"]), c=t(d.get("c")), dir=t(d.get("dir")))


class PlaneWaves:
    """Plane-wave mode table of the point path: sx, sy, zref (J,) float64; gamma (J,) complex128; p (J,3)."""

    def __init__(self, *, lam, sx, sy, gamma, zref, p, **_):
        self.lam, self.sx, self.sy, self.gamma, self.zref, self.p = float(lam), sx, sy, gamma, zref, p

    def struct(self):
        m = scw_modes()
        m.struct_size = ctypes.sizeof(scw_modes)
        m.kind = SCW_MODES_PLANEWAVE
        m.dtype = _dt(self.p)
        m.J = self.p.shape[0]
        m.lambda_ = self.lam
        m.sx, m.sy, m.gamma = self.sx.data_ptr(), self.sy.data_ptr(), self.gamma.data_ptr()
        m.zref, m.p = self.zref.data_ptr(), self.p.data_ptr()
        return m

    @staticmethod
    def from_numpy(d, device):
        t = lambda a: torch.from_numpy(a).to(device)
        return PlaneWaves(lam=d["lam"], sx=t(d["sx"]), sy=t(d["sy"]), gamma=t(d["gamma"]), zref=t(d["zref"]),
                          p=t(d["p"]))


class Exterior:
    """Half-space above (side=SCW_SIDE_ABOVE: incident + reflected) or below (transmitted) the sample, eq. 9.

    p_face, p_inc: (M, 3) complex device tensors (component fastest), p_inc None below / when there is no incident wave.
    """

    def __init__(self, *, side, U, Vn, X, Y, lam, n, z_face, p_face, z_inc=0.0, p_inc=None, **_):
        self.side, self.U, self.Vn, self.X, self.Y, self.lam = int(side), int(U), int(Vn), float(X), float(Y), float(lam)
        self.n, self.z_face, self.z_inc, self.p_face, self.p_inc = complex(n), float(z_face), float(z_inc), p_face, p_inc
        assert p_face.shape == (self.U * self.Vn, 3) and p_face.is_contiguous()
        assert p_inc is None or (p_inc.shape == p_face.shape and p_inc.dtype == p_face.dtype and p_inc.is_contiguous())

    def struct(self):
        return scw_exterior(ctypes.sizeof(scw_exterior), _dt(self.p_face), self.side, self.U, self.Vn, self.X, self.Y,
                            self.lam, self.n.real, self.n.imag, self.z_face, self.z_inc, self.p_face.data_ptr(),
                            None if self.p_inc is None else self.p_inc.data_ptr())

    @staticmethod
    def from_numpy(d, device):
        t = lambda a: None if a is None else torch.from_numpy(a).to(device)
        return Exterior(side=d["side"], U=d["U"], Vn=d["Vn"], X=d["X"], Y=d["Y"], lam=d["lam"], n=d["n"],
                        z_face=d["z_face"], z_inc=d.get("z_inc", 0.0), p_face=t(d["p_face"]), p_inc=t(d.get("p_inc")))


class Context:
    """scw_ctx bound to a torch device and stream; owns a growable torch workspace buffer."""

    def __init__(self, device=0, stream=None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2404_07293_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.device = torch.device("cuda", device) if isinstance(device, int) else torch.device(device)
        self.L = lib()
        self._h = c_void_p()
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.stream = st
        s = self.L.scw_create(byref(self._h), self.device.index or 0, c_void_p(st.cuda_stream))
        if s != 0:
            raise ScwError(s, "scw_create failed (device must be compute capability 10.x)")
        self._ws = None

    def close(self):
        if self._h:
            self.L.scw_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers
    def check(self, status):
        if status != 0:
            raise ScwError(status, self.L.scw_last_error(self._h).decode())

    def last_error(self):
        return self.L.scw_last_error(self._h).decode()

    def launch_count(self):
        return int(self.L.scw_launch_count(self._h))

    def last_kernels(self):
        """Names of the kernel classes the last hot-path call launched (scw_last_kernels)."""
        bits = int(self.L.scw_last_kernels(self._h))
        return [self.L.scw_profile_name(k).decode() for k in range(self.L.scw_profile_classes()) if (bits >> k) & 1]

    def set_path(self, path):
        self.check(self.L.scw_set_option(self._h, SCW_OPT_PATH, path))

    def set_cache(self, on):
        """SCW_OPT_CACHE: keep the twiddle tables in the workspace between consecutive sweep calls (see scwatter.h)."""
        self.check(self.L.scw_set_option(self._h, SCW_OPT_CACHE, 1 if on else 0))

    def invalidate_cache(self):
        self.check(self.L.scw_invalidate_cache(self._h))

    def set_profile(self, on):
        self.check(self.L.scw_set_option(self._h, SCW_OPT_PROFILE, 1 if on else 0))
        self.check(self.L.scw_profile_reset(self._h))

    def profile(self):
        """{kernel name: (device ms, launches)} accumulated since set_profile(True) / the last reset."""
        out = {}
        for kc in range(self.L.scw_profile_classes()):
            ms, n = c_double(), c_int64()
            self.check(self.L.scw_profile_read(self._h, kc, byref(ms), byref(n)))
            if n.value:
                out[self.L.scw_profile_name(kc).decode()] = (ms.value, n.value)
        return out

    def measure_peaks(self, reps=5, hbm_bytes=1 << 30):
        """{unit: measured rate} from the library's microbenchmarks (scw_measure_peak); synchronises the stream."""
        buf = torch.empty(int(hbm_bytes), dtype=torch.uint8, device=self.device)
        out = {}
        for name, which in SCW_PEAKS.items():
            v = c_double()
            self.check(self.L.scw_measure_peak(self._h, which, c_void_p(buf.data_ptr()), buf.numel(), reps, byref(v)))
            out[name] = v.value
        return out

    def assembly_timeline(self):
        """[(us to: own weights written, all weights seen, span streamed, exit)] per CTA of the last tcgen05 assembly."""
        buf = (c_double * (256 * 4))()
        n = c_int32()
        self.check(self.L.scw_profile_assembly(self._h, 256, buf, byref(n)))
        return [tuple(buf[4 * i:4 * i + 4]) for i in range(n.value)]

    def kernel_timeline(self, max_n=128):
        """[(exit_ns, kernel class name)] of the last tensor-core sweep launches, oldest first (scw_profile_timeline)."""
        ns = (ctypes.c_uint64 * max_n)()
        kc = (c_int32 * max_n)()
        n = c_int32()
        self.check(self.L.scw_profile_timeline(self._h, max_n, ns, kc, byref(n)))
        return [(int(ns[i]), self.L.scw_profile_name(kc[i]).decode()) for i in range(n.value)]

    def reserve(self, nbytes):
        """Grow the registered workspace to at least nbytes."""
        if nbytes and (self._ws is None or self._ws.numel() < nbytes):
            self._ws = None
            self._ws = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
            self.check(self.L.scw_set_workspace(self._h, c_void_p(self._ws.data_ptr()), self._ws.numel()))

    def workspace_bytes(self):
        return 0 if self._ws is None else self._ws.numel()


# ---------------------------------------------------------------------------------------------
def scw_assemble_spectra(ctx, layer, z, out=None):
    """P = V (c o g(z)): returns P as a (Fz, ldP) tensor (column-major [ldP x Fz])."""
    Fz = z.numel()
    st = layer.struct()
    need = c_size_t()
    ctx.check(ctx.L.scw_assemble_workspace(ctx._h, byref(st), Fz, byref(need)))
    ctx.reserve(need.value)
    if out is None:
        out = torch.empty((Fz, layer.R), dtype=layer.V.dtype, device=ctx.device)
    ctx.check(ctx.L.scw_assemble_spectra(ctx._h, byref(st), Fz, _p(z), _p(out), out.shape[1] if Fz else layer.R))
    return out


def scw_synthesize_grid(ctx, *, U, Vn, X, Y, P, x, y, out=None, strides=None):
    """E[n, comp, k, i] = sum_uv P[n, comp*M+m] exp(i 2 pi (u x_i/X + v y_k/Y)); P is (Fz, ldP)."""
    Fz, Nx, Ny = P.shape[0], x.numel(), y.numel()
    dt = _dt(P)
    need = c_size_t()
    ctx.check(ctx.L.scw_synthesize_workspace(ctx._h, dt, U, Vn, Fz, Nx, Ny, byref(need)))
    ctx.reserve(need.value)
    if out is None:
        out = torch.empty((Fz, 3, Ny, Nx), dtype=P.dtype, device=ctx.device)
    sarr = None if strides is None else (c_int64 * 4)(*strides)
    ctx.check(ctx.L.scw_synthesize_grid(ctx._h, dt, U, Vn, X, Y, Fz, _p(P), P.shape[1], Nx, _p(x), Ny, _p(y),
                                        _p(out), sarr))
    return out


def scw_eval_points(ctx, modes, r, out=None):
    """E (N, 3) at points r (N, 3) float64; modes is a PlaneWaves table or a Layer (dense eq. 34)."""
    N = r.shape[0]
    if isinstance(modes, Layer):
        m = scw_modes()
        m.struct_size = ctypes.sizeof(scw_modes)
        m.kind = SCW_MODES_DENSE
        m.layer = modes.struct()
        dtype = modes.V.dtype
    else:
        m = modes.struct()
        dtype = modes.p.dtype
    need = c_size_t()
    ctx.check(ctx.L.scw_points_workspace(ctx._h, byref(m), N, byref(need)))
    ctx.reserve(need.value)
    if out is None:
        out = torch.empty((N, 3), dtype=dtype, device=ctx.device)
    ctx.check(ctx.L.scw_eval_points(ctx._h, byref(m), N, _p(r), _p(out)))
    return out


SCW_POINTS_NOALLOC_MAX_J = 8192


def scw_eval_points_noalloc(ctx, modes, r, out):
    """scw_eval_points for a caller that cannot allocate GPU memory (a plug-in inside an application whose pool owns the
    whole device, a real-time loop that must stay off the allocator, an out-of-memory handler): the plane-wave table
    goes into an array built into libscw.so instead of a workspace, so neither the library nor this wrapper allocates
    anything -- `out` (N, 3) is required and must be the caller's own tensor.  modes: a PlaneWaves table with at most
    SCW_POINTS_NOALLOC_MAX_J waves for complex64 (more is refused with ScwError, status 2).  All callers on one GPU share
    that array: do not let two of these calls overlap on the device.  Make the first call per device at start-up."""
    if isinstance(modes, Layer):
        raise ScwError(8, "scw_eval_points_noalloc takes a PlaneWaves table, not a Layer")
    if out is None:
        raise ScwError(1, "scw_eval_points_noalloc: pass the output tensor (this call allocates nothing)")
    m = modes.struct()
    ctx.check(ctx.L.scw_eval_points_noalloc(ctx._h, byref(m), r.shape[0], _p(r), _p(out)))
    return out


def scw_exterior_spectra(ctx, ext, z, out=None):
    """eq. 9 on the planes z: P as a (Fz, 3M) tensor (column-major [3M x Fz]); feed it to scw_synthesize_grid."""
    Fz, R = z.numel(), 3 * ext.U * ext.Vn
    st = ext.struct()
    if out is None:
        out = torch.empty((Fz, R), dtype=ext.p_face.dtype, device=ctx.device)
    ctx.check(ctx.L.scw_exterior_spectra(ctx._h, byref(st), Fz, _p(z), _p(out), out.shape[1] if Fz else R))
    return out


def scw_exterior_grid(ctx, ext, z, x, y, out=None, strides=None):
    """eq. 9-10 on a rectilinear grid in one call: E (Fz, 3, Ny, Nx)."""
    Fz, Nx, Ny = z.numel(), x.numel(), y.numel()
    st = ext.struct()
    need = c_size_t()
    ctx.check(ctx.L.scw_exterior_grid_workspace(ctx._h, byref(st), Fz, Nx, Ny, byref(need)))
    ctx.reserve(need.value)
    if out is None:
        out = torch.empty((Fz, 3, Ny, Nx), dtype=ext.p_face.dtype, device=ctx.device)
    sarr = None if strides is None else (c_int64 * 4)(*strides)
    ctx.check(ctx.L.scw_exterior_grid(ctx._h, byref(st), Fz, _p(z), Nx, _p(x), Ny, _p(y), _p(out), sarr))
    return out


def scw_exterior_points(ctx, ext, r, out=None):
    """eq. 9-10 at scattered points r (N, 3) float64 -> E (N, 3)."""
    N = r.shape[0]
    st = ext.struct()
    need = c_size_t()
    ctx.check(ctx.L.scw_exterior_points_workspace(ctx._h, byref(st), N, byref(need)))
    ctx.reserve(need.value)
    if out is None:
        out = torch.empty((N, 3), dtype=ext.p_face.dtype, device=ctx.device)
    ctx.check(ctx.L.scw_exterior_points(ctx._h, byref(st), N, _p(r), _p(out)))
    return out


def _sweep_args(layers, zs):
    n = len(layers)
    inst = (scw_layer * max(n, 1))(*[l._cached_struct() for l in layers])
    Fz = (c_int64 * max(n, 1))(*[z.numel() for z in zs])
    zp = (c_void_p * max(n, 1))(*[z.data_ptr() for z in zs])
    return n, inst, Fz, zp


def scw_sweep_wavelengths(ctx, layers, zs, x, y, out=None, strides=None):
    """Assembly + synthesis for every (wavelength, layer) instance; returns a list of E tensors."""
    n, inst, Fz, zp = _sweep_args(layers, zs)
    Nx, Ny = x.numel(), y.numel()
    need = c_size_t()
    ctx.check(ctx.L.scw_sweep_workspace(ctx._h, n, inst, Fz, Nx, Ny, byref(need)))
    ctx.reserve(need.value)
    if out is None:
        out = [torch.empty((z.numel(), 3, Ny, Nx), dtype=l.V.dtype, device=ctx.device) for l, z in zip(layers, zs)]
    Ep = (c_void_p * max(n, 1))(*[e.data_ptr() for e in out])
    sarr = None if strides is None else (c_int64 * 4)(*strides)
    ctx.check(ctx.L.scw_sweep_wavelengths(ctx._h, n, inst, Fz, zp, Nx, _p(x), Ny, _p(y), Ep, sarr))
    return out


def scw_calibrate(ctx, layers, zs, x, y, out=None, strides=None, reps=5):
    """Calibrate the stream-K split of the tensor-core assembly by running this sweep (synchronises); returns E."""
    n, inst, Fz, zp = _sweep_args(layers, zs)
    Nx, Ny = x.numel(), y.numel()
    need = c_size_t()
    ctx.check(ctx.L.scw_sweep_workspace(ctx._h, n, inst, Fz, Nx, Ny, byref(need)))
    ctx.reserve(need.value)
    if out is None:
        out = [torch.empty((z.numel(), 3, Ny, Nx), dtype=l.V.dtype, device=ctx.device) for l, z in zip(layers, zs)]
    Ep = (c_void_p * max(n, 1))(*[e.data_ptr() for e in out])
    sarr = None if strides is None else (c_int64 * 4)(*strides)
    ctx.check(ctx.L.scw_calibrate(ctx._h, n, inst, Fz, zp, Nx, _p(x), Ny, _p(y), Ep, sarr, reps))
    return out


def scw_sweep_intensity(ctx, layers, zs, x, y, out=None, strides=None):
    """Detector intensity I = sum_comp |E_comp|^2 of every instance (real tensors [Fz, Ny, Nx]); E is never stored."""
    n, inst, Fz, zp = _sweep_args(layers, zs)
    Nx, Ny = x.numel(), y.numel()
    need = c_size_t()
    ctx.check(ctx.L.scw_sweep_intensity_workspace(ctx._h, n, inst, Fz, Nx, Ny, byref(need)))
    ctx.reserve(need.value)
    if out is None:
        real = {torch.complex64: torch.float32, torch.complex128: torch.float64}
        out = [torch.empty((z.numel(), Ny, Nx), dtype=real[l.V.dtype], device=ctx.device) for l, z in zip(layers, zs)]
    Ip = (c_void_p * max(n, 1))(*[e.data_ptr() for e in out])
    sarr = None if strides is None else (c_int64 * 3)(*strides)
    ctx.check(ctx.L.scw_sweep_intensity(ctx._h, n, inst, Fz, zp, Nx, _p(x), Ny, _p(y), Ip, sarr))
    return out


def scw_sweep_detector(ctx, layers, zs, x, y, window=None, want_I=True, want_S=True, out_I=None, out_S=None, strides=None):
    """Detector reductions of a sweep: (I list or None, S list or None).  I[i]: [Fz, Ny, Nx] intensity, S[i]: [Fz] sums
    of I over the window (ix0, ix1, iy0, iy1) of grid indices (None = whole plane); the complex field is never stored."""
    n, inst, Fz, zp = _sweep_args(layers, zs)
    Nx, Ny = x.numel(), y.numel()
    need = c_size_t()
    ctx.check(ctx.L.scw_sweep_detector_workspace(ctx._h, n, inst, Fz, Nx, Ny, byref(need)))
    ctx.reserve(need.value)
    real = {torch.complex64: torch.float32, torch.complex128: torch.float64}
    if want_I and out_I is None:
        out_I = [torch.empty((z.numel(), Ny, Nx), dtype=real[l.V.dtype], device=ctx.device) for l, z in zip(layers, zs)]
    if want_S and out_S is None:
        out_S = [torch.empty((z.numel(),), dtype=real[l.V.dtype], device=ctx.device) for l, z in zip(layers, zs)]
    Ip = (c_void_p * max(n, 1))(*[e.data_ptr() for e in out_I]) if want_I else None
    Sp = (c_void_p * max(n, 1))(*[e.data_ptr() for e in out_S]) if want_S else None
    sarr = None if strides is None else (c_int64 * 3)(*strides)
    w = None if window is None else byref(scw_window(*[int(v) for v in window]))
    ctx.check(ctx.L.scw_sweep_detector(ctx._h, n, inst, Fz, zp, Nx, _p(x), Ny, _p(y), Ip, sarr, w, Sp))
    return (out_I if want_I else None), (out_S if want_S else None)


def scw_absorbance(ctx, S, S0, w=None, want_band=False):
    """A = -log10(S / S0) elementwise; with want_band also -log10(sum w S / sum w S0) as a 1-element tensor."""
    dt = SCW_C64 if S.dtype == torch.float32 else SCW_C128
    A = torch.empty_like(S)
    band = torch.empty((1,), dtype=S.dtype, device=S.device) if want_band else None
    ctx.check(ctx.L.scw_absorbance(ctx._h, dt, S.numel(), _p(S), _p(S0), _p(w), _p(A), _p(band)))
    return (A, band) if want_band else A


def scw_build_V(ctx, *, U, Vn, X, Y, lam, Q, psi, alpha=None, out=None, ldV=None):
    """V = T Q [diag(alpha)] (eq. 33): Q (J, ldQ) complex (column-major [ldQ x J], rows P_x, P_y, B_x, B_y), psi (M,),
    alpha (J,) or None.  Returns V as a (J, ldV) tensor (column-major [ldV x J])."""
    J, ldQ = Q.shape
    M = U * Vn
    vb = scw_vbuild(ctypes.sizeof(scw_vbuild), _dt(Q), U, Vn, X, Y, lam, J, Q.data_ptr(), ldQ, psi.data_ptr(),
                    None if alpha is None else alpha.data_ptr())
    need = c_size_t()
    ctx.check(ctx.L.scw_build_V_workspace(ctx._h, byref(vb), byref(need)))
    ctx.reserve(need.value)
    if out is None:
        out = torch.zeros((J, 3 * M if ldV is None else ldV), dtype=Q.dtype, device=ctx.device)
    ctx.check(ctx.L.scw_build_V(ctx._h, byref(vb), _p(out), out.shape[1]))
    return out


def scw_propagate_alpha(ctx, *, lam, z_if, Q, gamma, r0, dir=None, want_rL=True):
    """alpha^(l) of every layer (eq. 24-26).  Q: list of (n, ldQ) complex device tensors (column-major [ldQ x n]: row j of
    the tensor is column j = mode j of Q), gamma: list of (n,) complex128, dir: list of (n,) int8 or None, z_if: L + 1
    floats (host), r0: (n,) field vector at z_0.  Returns (list of alpha tensors, r_L or None)."""
    L_ = len(Q)
    n, ldQ = Q[0].shape
    zarr = (c_double * (L_ + 1))(*[float(v) for v in z_if])
    Qp = (c_void_p * L_)(*[q.data_ptr() for q in Q])
    gp = (c_void_p * L_)(*[g.data_ptr() for g in gamma])
    dp = None if dir is None else (c_void_p * L_)(*[d.data_ptr() for d in dir])
    st = scw_stack(ctypes.sizeof(scw_stack), _dt(Q[0]), L_, n, float(lam), zarr, Qp, ldQ, gp, dp)
    need = c_size_t()
    ctx.check(ctx.L.scw_propagate_alpha_workspace(ctx._h, byref(st), byref(need)))
    ctx.reserve(need.value)
    alphas = [torch.empty((n,), dtype=Q[0].dtype, device=ctx.device) for _ in range(L_)]
    ap = (c_void_p * L_)(*[a.data_ptr() for a in alphas])
    rL = torch.empty((n,), dtype=Q[0].dtype, device=ctx.device) if want_rL else None
    ctx.check(ctx.L.scw_propagate_alpha(ctx._h, byref(st), _p(r0), ap, _p(rL)))
    return alphas, rL


def scw_sweep_wavelengths_host(ctx, layers, zs, x, y, out=None):
    """Host-buffer variant: every tensor lives in (pinned) host memory; returns (E list, h2d, d2h bytes)."""
    n, inst, Fz, zp = _sweep_args(layers, zs)
    Nx, Ny = x.numel(), y.numel()
    need = c_size_t()
    ctx.check(ctx.L.scw_sweep_host_workspace(ctx._h, n, inst, Fz, Nx, Ny, byref(need)))
    ctx.reserve(need.value)
    if out is None:
        out = [torch.empty((z.numel(), 3, Ny, Nx), dtype=l.V.dtype).pin_memory() for l, z in zip(layers, zs)]
    Ep = (c_void_p * max(n, 1))(*[e.data_ptr() for e in out])
    up, down = c_int64(), c_int64()
    ctx.check(ctx.L.scw_sweep_wavelengths_host(ctx._h, n, inst, Fz, zp, Nx, _p(x), Ny, _p(y), Ep, byref(up),
                                               byref(down)))
    return out, up.value, down.value
