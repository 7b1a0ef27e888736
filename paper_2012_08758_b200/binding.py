"""Thin ctypes binding of libac_mhd.so (include/ac_mhd.h).  Argument marshalling only: every step
of the path runs in the library's CUDA kernels.  There is no fallback: if the library is missing
or a call fails, this raises.

PyTorch is used for device memory (the workspace tensor) and streams only.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libac_mhd.so")

AC_F32, AC_F64 = 0, 1
AC_PART_INNER, AC_PART_OUTER = 1, 2
NFIELDS = 7
EXPORTS = (
    "ac_workspace_bytes", "ac_init", "ac_load_state", "ac_store_state", "ac_load_field", "ac_store_field", "ac_step",
    "ac_reduce",
    "ac_forcing_from_draws", "ac_forcing_params", "ac_make_forcing", "ac_set_bext", "ac_set_cfl", "ac_set_variant",
    "ac_set_upwind", "ac_set_mixed", "ac_substep", "ac_state_layout", "ac_field_device_ptr", "ac_reduce_raw",
    "ac_reduce_ext", "ac_reduce_ext_raw", "ac_set_slab", "ac_substep_part", "ac_halo_bytes", "ac_halo_pack",
    "ac_halo_unpack", "ac_diag_combine", "ac_set_forcing_mode", "ac_halo_pull", "ac_workspace_ptr", "ac_ipc_export",
    "ac_ipc_open", "ac_ipc_close", "ac_reduce_dense_noalloc", "ac_noalloc_max_cells",
    "ac_launch_count", "ac_free", "ac_strerror", "ac_version",
)


class AcGrid(ctypes.Structure):
    _fields_ = [("nx", ctypes.c_int), ("ny", ctypes.c_int), ("nz", ctypes.c_int),
                ("lx", ctypes.c_double), ("ly", ctypes.c_double), ("lz", ctypes.c_double)]


class AcLayoutInfo(ctypes.Structure):
    _fields_ = [("elem_bytes", ctypes.c_int), ("packed_pairs", ctypes.c_int), ("gx", ctypes.c_int),
                ("pitch", ctypes.c_int), ("my", ctypes.c_int), ("mz", ctypes.c_int),
                ("plane_elems", ctypes.c_size_t), ("field_elems", ctypes.c_size_t)]


class AcForcing(ctypes.Structure):
    _fields_ = [("k", ctypes.c_double * 3), ("phase", ctypes.c_double),
                ("re", ctypes.c_double * 3), ("im", ctypes.c_double * 3)]

    def as_tuple(self):
        return (np.array(self.k[:]), float(self.phase), np.array(self.re[:]), np.array(self.im[:]))

    @classmethod
    def from_tuple(cls, t):
        k, phase, re, im = t
        f = cls()
        f.k[:] = [float(v) for v in k]
        f.phase = float(phase)
        f.re[:] = [float(v) for v in re]
        f.im[:] = [float(v) for v in im]
        return f


class AcDiag(ctypes.Structure):
    _fields_ = [("urms", ctypes.c_double), ("umax", ctypes.c_double), ("brms", ctypes.c_double),
                ("bmax", ctypes.c_double), ("lnrho_min", ctypes.c_double), ("lnrho_max", ctypes.c_double),
                ("dt_cfl", ctypes.c_double), ("nonfinite", ctypes.c_int)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class AcDiagExt(ctypes.Structure):
    _fields_ = [("kin_hel", ctypes.c_double), ("cur_hel", ctypes.c_double), ("va_max", ctypes.c_double),
                ("dt_cfl_alfven", ctypes.c_double), ("nonfinite", ctypes.c_int)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class AcError(RuntimeError):
    pass


_lib = None


def load_library():
    """dlopen the in-tree library and declare the signatures.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise AcError("libac_mhd.so not built: run `python -m paper_2012_08758_b200.build` "
                      "(or __graft_entry__.build()); there is no CPU fallback")
    L = ctypes.CDLL(LIB_PATH)
    vp, dbl, i32 = ctypes.c_void_p, ctypes.c_double, ctypes.c_int
    L.ac_workspace_bytes.argtypes = [ctypes.POINTER(AcGrid), i32]
    L.ac_workspace_bytes.restype = ctypes.c_size_t
    L.ac_init.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(AcGrid), i32, dbl, dbl, dbl, dbl, dbl, vp, vp]
    L.ac_load_state.argtypes = [vp, ctypes.POINTER(vp), i32]
    L.ac_store_state.argtypes = [vp, ctypes.POINTER(vp), i32]
    L.ac_load_field.argtypes = [vp, i32, vp, i32]
    L.ac_store_field.argtypes = [vp, i32, vp, i32]
    L.ac_step.argtypes = [vp, dbl, ctypes.POINTER(AcForcing)]
    L.ac_reduce.argtypes = [vp, ctypes.POINTER(AcDiag)]
    L.ac_forcing_from_draws.argtypes = [vp, dbl, dbl, dbl, dbl, dbl, ctypes.POINTER(AcForcing)]
    L.ac_forcing_params.argtypes = [dbl, dbl, dbl, ctypes.POINTER(AcGrid), dbl, dbl, dbl, dbl, dbl,
                                    ctypes.POINTER(AcForcing)]
    L.ac_make_forcing.argtypes = [vp, ctypes.c_uint64, ctypes.c_uint64, dbl, dbl, ctypes.POINTER(AcForcing)]
    L.ac_set_bext.argtypes = [vp, ctypes.POINTER(dbl)]
    L.ac_set_cfl.argtypes = [vp, dbl, dbl]
    L.ac_set_variant.argtypes = [vp, i32]
    L.ac_set_upwind.argtypes = [vp, i32]
    L.ac_set_upwind.restype = i32
    L.ac_set_mixed.argtypes = [vp, i32]
    L.ac_set_mixed.restype = i32
    L.ac_substep.argtypes = [vp, i32, dbl, ctypes.POINTER(AcForcing)]
    L.ac_substep.restype = i32
    L.ac_state_layout.argtypes = [vp, ctypes.POINTER(AcLayoutInfo)]
    L.ac_state_layout.restype = i32
    L.ac_field_device_ptr.argtypes = [vp, i32]
    L.ac_field_device_ptr.restype = ctypes.c_void_p
    L.ac_reduce_raw.argtypes = [vp, ctypes.POINTER(dbl)]
    L.ac_reduce_raw.restype = i32
    L.ac_reduce_ext.argtypes = [vp, ctypes.POINTER(AcDiagExt)]
    L.ac_reduce_ext.restype = i32
    L.ac_reduce_ext_raw.argtypes = [vp, ctypes.POINTER(dbl)]
    L.ac_reduce_ext_raw.restype = i32
    L.ac_halo_pull.argtypes = [vp, vp, vp, vp]
    L.ac_halo_pull.restype = i32
    L.ac_workspace_ptr.argtypes = [vp]
    L.ac_workspace_ptr.restype = ctypes.c_void_p
    L.ac_ipc_export.argtypes = [vp, vp]
    L.ac_ipc_export.restype = i32
    L.ac_ipc_open.argtypes = [vp, ctypes.POINTER(vp)]
    L.ac_ipc_open.restype = i32
    L.ac_ipc_close.argtypes = [vp]
    L.ac_ipc_close.restype = i32
    L.ac_set_forcing_mode.argtypes = [vp, i32]
    L.ac_set_forcing_mode.restype = i32
    L.ac_set_slab.argtypes = [vp, i32, i32]
    L.ac_set_slab.restype = i32
    L.ac_substep_part.argtypes = [vp, i32, dbl, ctypes.POINTER(AcForcing), i32]
    L.ac_substep_part.restype = i32
    L.ac_halo_bytes.argtypes = [vp]
    L.ac_halo_bytes.restype = ctypes.c_size_t
    L.ac_halo_pack.argtypes = [vp, vp, vp, vp]
    L.ac_halo_pack.restype = i32
    L.ac_halo_unpack.argtypes = [vp, vp, vp, vp]
    L.ac_halo_unpack.restype = i32
    L.ac_diag_combine.argtypes = [vp, ctypes.POINTER(dbl), i32, ctypes.POINTER(AcDiag)]
    L.ac_diag_combine.restype = i32
    L.ac_reduce_dense_noalloc.argtypes = [vp, i32, ctypes.POINTER(AcGrid), ctypes.POINTER(dbl), vp, vp]
    L.ac_reduce_dense_noalloc.restype = i32
    L.ac_noalloc_max_cells.argtypes = []
    L.ac_noalloc_max_cells.restype = ctypes.c_longlong
    L.ac_launch_count.argtypes = [vp]
    L.ac_launch_count.restype = ctypes.c_longlong
    L.ac_free.argtypes = [vp]
    L.ac_free.restype = None
    L.ac_strerror.argtypes = [i32]
    L.ac_strerror.restype = ctypes.c_char_p
    L.ac_version.restype = ctypes.c_char_p
    for name in ("ac_init", "ac_load_state", "ac_store_state", "ac_load_field", "ac_store_field", "ac_step", "ac_reduce", "ac_forcing_from_draws",
                 "ac_forcing_params", "ac_make_forcing", "ac_set_bext", "ac_set_cfl", "ac_set_variant"):
        getattr(L, name).restype = i32
    _lib = L
    return L


def _check(rc, what):
    if rc != 0:
        raise AcError("%s failed: %s (%d)" % (what, load_library().ac_strerror(rc).decode(), rc))


def _grid(shape, lengths):
    nz, ny, nx = shape
    return AcGrid(int(nx), int(ny), int(nz), float(lengths[0]), float(lengths[1]), float(lengths[2]))


def ac_workspace_bytes(shape, lengths, dtype):
    g = _grid(shape, lengths)
    return int(load_library().ac_workspace_bytes(ctypes.byref(g), int(dtype)))


def ac_forcing_params(k_f, helicity, cs, shape, lengths, u1, u2, u3, dt, f0):
    """Host-only Eq. 4-6 helper (no device needed)."""
    g = _grid(shape, lengths)
    f = AcForcing()
    _check(load_library().ac_forcing_params(float(k_f), float(helicity), float(cs), ctypes.byref(g), float(u1),
                                            float(u2), float(u3), float(dt), float(f0), ctypes.byref(f)),
           "ac_forcing_params")
    return f


def ac_ipc_open(handle):
    """Maps a workspace another process exported with Context.ac_ipc_export; returns its device address here."""
    out = ctypes.c_void_p()
    _check(load_library().ac_ipc_open(ctypes.c_char_p(handle), ctypes.byref(out)), "ac_ipc_open")
    return int(out.value)


def ac_ipc_close(ptr):
    _check(load_library().ac_ipc_close(ctypes.c_void_p(ptr)), "ac_ipc_close")


def ac_noalloc_max_cells():
    return int(load_library().ac_noalloc_max_cells())


def ac_reduce_dense_noalloc(state, lengths, raw_out, bext=None, stream=None):
    """The reductions of ac_reduce_raw of a dense DEVICE state (torch CUDA tensor (7, nz, ny, nx), float32 or float64,
    contiguous) into raw_out (torch CUDA tensor of 6 float64), without a context and without any allocation inside the
    library (include/ac_mhd.h: at most ac_noalloc_max_cells() cells, calls must not overlap on the GPU).  Launches on
    `stream` (a torch stream; None: torch's current stream) and returns without synchronising.  Marshalling only."""
    import torch
    if not (isinstance(state, torch.Tensor) and isinstance(raw_out, torch.Tensor) and state.is_cuda and raw_out.is_cuda):
        raise AcError("ac_reduce_dense_noalloc takes CUDA tensors (no CPU fallback)")
    if state.dim() != 4 or state.shape[0] != 7 or not state.is_contiguous():
        raise AcError("state must be a contiguous (7, nz, ny, nx) tensor")
    if state.dtype not in (torch.float32, torch.float64):
        raise AcError("state must be float32 or float64")
    if raw_out.dtype != torch.float64 or raw_out.numel() != 6 or not raw_out.is_contiguous():
        raise AcError("raw_out must be 6 contiguous float64")
    if raw_out.device != state.device:
        raise AcError("state and raw_out must live on the same device")
    grid = _grid(tuple(state.shape[1:]), lengths)
    dtype = AC_F64 if state.dtype == torch.float64 else AC_F32
    b = (ctypes.c_double * 3)(*[float(v) for v in bext]) if bext is not None else None
    with torch.cuda.device(state.device):
        st = stream if stream is not None else torch.cuda.current_stream(state.device)
        _check(load_library().ac_reduce_dense_noalloc(ctypes.c_void_p(state.data_ptr()), dtype, ctypes.byref(grid), b,
                                                      ctypes.c_void_p(raw_out.data_ptr()),
                                                      ctypes.c_void_p(st.cuda_stream)), "ac_reduce_dense_noalloc")


def ac_version():
    return load_library().ac_version().decode()


class Context:
    """One ac_ctx.  Methods carry the C names: ac_load_state, ac_step, ac_reduce, ..."""

    def __init__(self, shape, lengths=(2 * np.pi,) * 3, dtype=AC_F64, nu=0.0, eta=0.0, cs=1.0, k_f=3.0,
                 helicity=0.0, stream=None, device="cuda:0", own_workspace=False):
        import torch          # device memory and streams only
        L = load_library()
        if not torch.cuda.is_available():
            raise AcError("no CUDA device: the MHD path runs only on the GPU (no CPU fallback)")
        self.shape = tuple(int(s) for s in shape)
        self.lengths = tuple(float(v) for v in lengths)
        self.dtype = int(dtype)
        self.np_dtype = np.float64 if self.dtype == AC_F64 else np.float32
        self.torch_dtype = torch.float64 if self.dtype == AC_F64 else torch.float32
        self.device = torch.device(device)
        g = _grid(self.shape, self.lengths)
        nbytes = L.ac_workspace_bytes(ctypes.byref(g), self.dtype)
        if nbytes == 0:
            raise AcError("invalid grid %r" % (self.shape,))
        with torch.cuda.device(self.device):
            # own_workspace: the library cudaMallocs the workspace itself (needed for ac_ipc_export)
            self.workspace = None if own_workspace else torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        base = self.workspace.data_ptr() if self.workspace is not None else 0
        aligned = (base + 255) // 256 * 256
        self._ctx = ctypes.c_void_p()
        with torch.cuda.device(self.device):       # the library records the current device as the context's
            rc = L.ac_init(ctypes.byref(self._ctx), ctypes.byref(g), self.dtype, float(nu), float(eta), float(cs),
                           float(k_f), float(helicity), ctypes.c_void_p(aligned),
                           ctypes.c_void_p(self.stream.cuda_stream))
        _check(rc, "ac_init")
        self._lib = L

    # -- marshalling helpers --------------------------------------------------------------------
    def _ptr_array(self, ptrs):
        arr = (ctypes.c_void_p * NFIELDS)()
        for i, p in enumerate(ptrs):
            arr[i] = p
        return arr

    # -- C ABI ----------------------------------------------------------------------------------
    def ac_load_state(self, state):
        """state: numpy (7, nz, ny, nx) or torch tensor (host, pinned host, or device)."""
        import torch
        if isinstance(state, np.ndarray):
            st = np.ascontiguousarray(state, dtype=self.np_dtype)
            assert st.shape == (NFIELDS,) + self.shape
            self._keep = st
            ptrs = [st[q].ctypes.data for q in range(NFIELDS)]
            on_dev = 0
        else:
            assert state.dtype == self.torch_dtype and state.is_contiguous()
            assert tuple(state.shape) == (NFIELDS,) + self.shape
            self._keep = state
            ptrs = [state[q].data_ptr() for q in range(NFIELDS)]
            on_dev = 1 if state.is_cuda else 0
        _check(self._lib.ac_load_state(self._ctx, self._ptr_array(ptrs), on_dev), "ac_load_state")
        if not on_dev and isinstance(state, np.ndarray):
            self.synchronize()          # pageable numpy memory: do not let the caller race the copy

    def ac_store_state(self, out=None):
        """Returns the state as numpy (7, nz, ny, nx), or fills `out` (numpy / torch host or device)."""
        if out is None:
            out = np.empty((NFIELDS,) + self.shape, dtype=self.np_dtype)
        if isinstance(out, np.ndarray):
            assert out.dtype == self.np_dtype and out.flags["C_CONTIGUOUS"]
            ptrs = [out[q].ctypes.data for q in range(NFIELDS)]
            on_dev = 0
        else:
            assert out.dtype == self.torch_dtype and out.is_contiguous()
            ptrs = [out[q].data_ptr() for q in range(NFIELDS)]
            on_dev = 1 if out.is_cuda else 0
        _check(self._lib.ac_store_state(self._ctx, self._ptr_array(ptrs), on_dev), "ac_store_state")
        return out

    def _field_ptr(self, arr):
        if isinstance(arr, np.ndarray):
            assert arr.dtype == self.np_dtype and arr.flags["C_CONTIGUOUS"] and arr.shape == self.shape
            return arr.ctypes.data, 0
        assert arr.dtype == self.torch_dtype and arr.is_contiguous() and tuple(arr.shape) == self.shape
        return arr.data_ptr(), (1 if arr.is_cuda else 0)

    def ac_load_field(self, q, field):
        """field: numpy (nz, ny, nx) or torch tensor (host or device) of the context's dtype."""
        ptr, on_dev = self._field_ptr(field)
        _check(self._lib.ac_load_field(self._ctx, int(q), ctypes.c_void_p(ptr), on_dev), "ac_load_field")
        if not on_dev:
            self.synchronize()

    def ac_store_field(self, q, out):
        ptr, on_dev = self._field_ptr(out)
        _check(self._lib.ac_store_field(self._ctx, int(q), ctypes.c_void_p(ptr), on_dev), "ac_store_field")
        return out

    def ac_step(self, dt, forcing=None):
        f = None
        if forcing is not None:
            f = forcing if isinstance(forcing, AcForcing) else AcForcing.from_tuple(forcing)
        _check(self._lib.ac_step(self._ctx, float(dt), ctypes.byref(f) if f is not None else None), "ac_step")

    def ac_substep(self, s, dt, forcing=None):
        f = None
        if forcing is not None:
            f = forcing if isinstance(forcing, AcForcing) else AcForcing.from_tuple(forcing)
        _check(self._lib.ac_substep(self._ctx, int(s), float(dt), ctypes.byref(f) if f is not None else None),
               "ac_substep")

    def ac_substep_part(self, s, dt, forcing, part):
        f = None
        if forcing is not None:
            f = forcing if isinstance(forcing, AcForcing) else AcForcing.from_tuple(forcing)
        _check(self._lib.ac_substep_part(self._ctx, int(s), float(dt), ctypes.byref(f) if f is not None else None,
                                         int(part)), "ac_substep_part")

    def ac_set_slab(self, z0_plane, nz_global):
        _check(self._lib.ac_set_slab(self._ctx, int(z0_plane), int(nz_global)), "ac_set_slab")

    def ac_halo_bytes(self):
        return int(self._lib.ac_halo_bytes(self._ctx))

    def ac_halo_pack(self, send_lo, send_hi, stream=None):
        """send_lo / send_hi: device tensors of ac_halo_bytes() bytes each; stream: a torch stream or None."""
        _check(self._lib.ac_halo_pack(self._ctx, ctypes.c_void_p(send_lo.data_ptr()), ctypes.c_void_p(send_hi.data_ptr()),
                                      ctypes.c_void_p(stream.cuda_stream if stream is not None else 0)), "ac_halo_pack")

    def ac_halo_unpack(self, recv_lo, recv_hi, stream=None):
        _check(self._lib.ac_halo_unpack(self._ctx, ctypes.c_void_p(recv_lo.data_ptr()), ctypes.c_void_p(recv_hi.data_ptr()),
                                        ctypes.c_void_p(stream.cuda_stream if stream is not None else 0)), "ac_halo_unpack")

    def ac_halo_pull(self, below_workspace, above_workspace, stream=None):
        """below_workspace / above_workspace: integer device addresses (ac_workspace_ptr or ac_ipc_open)."""
        _check(self._lib.ac_halo_pull(self._ctx, ctypes.c_void_p(below_workspace), ctypes.c_void_p(above_workspace),
                                      ctypes.c_void_p(stream.cuda_stream if stream is not None else 0)), "ac_halo_pull")

    def ac_workspace_ptr(self):
        return int(self._lib.ac_workspace_ptr(self._ctx))

    def ac_ipc_export(self):
        buf = ctypes.create_string_buffer(64)
        _check(self._lib.ac_ipc_export(self._ctx, buf), "ac_ipc_export")
        return buf.raw

    def ac_diag_combine(self, raws):
        """raws: sequence of ac_reduce_raw tuples, one per rank, in rank order."""
        flat = (ctypes.c_double * (6 * len(raws)))(*[float(v) for r in raws for v in r])
        d = AcDiag()
        _check(self._lib.ac_diag_combine(self._ctx, flat, len(raws), ctypes.byref(d)), "ac_diag_combine")
        return d.as_dict()

    def ac_state_layout(self):
        info = AcLayoutInfo()
        _check(self._lib.ac_state_layout(self._ctx, ctypes.byref(info)), "ac_state_layout")
        return info

    def ac_field_device_ptr(self, q):
        p = self._lib.ac_field_device_ptr(self._ctx, int(q))
        if not p:
            raise AcError("ac_field_device_ptr failed")
        return int(p)

    def ac_reduce_raw(self):
        out = (ctypes.c_double * 6)()
        _check(self._lib.ac_reduce_raw(self._ctx, out), "ac_reduce_raw")
        return tuple(out)

    def ac_reduce(self):
        d = AcDiag()
        _check(self._lib.ac_reduce(self._ctx, ctypes.byref(d)), "ac_reduce")
        return d.as_dict()

    def ac_reduce_ext(self):
        d = AcDiagExt()
        _check(self._lib.ac_reduce_ext(self._ctx, ctypes.byref(d)), "ac_reduce_ext")
        return d.as_dict()

    def ac_reduce_ext_raw(self):
        out = (ctypes.c_double * 3)()
        _check(self._lib.ac_reduce_ext_raw(self._ctx, out), "ac_reduce_ext_raw")
        return tuple(out)

    def ac_forcing_from_draws(self, u1, u2, u3, dt, f0):
        f = AcForcing()
        _check(self._lib.ac_forcing_from_draws(self._ctx, float(u1), float(u2), float(u3), float(dt), float(f0),
                                               ctypes.byref(f)), "ac_forcing_from_draws")
        return f

    def ac_make_forcing(self, seed, step, dt, f0):
        f = AcForcing()
        _check(self._lib.ac_make_forcing(self._ctx, int(seed), int(step), float(dt), float(f0), ctypes.byref(f)),
               "ac_make_forcing")
        return f

    def ac_set_bext(self, b):
        arr = (ctypes.c_double * 3)(*[float(v) for v in b])
        _check(self._lib.ac_set_bext(self._ctx, arr), "ac_set_bext")

    def ac_set_cfl(self, c_u, c_nu):
        _check(self._lib.ac_set_cfl(self._ctx, float(c_u), float(c_nu)), "ac_set_cfl")

    def ac_set_variant(self, variant):
        _check(self._lib.ac_set_variant(self._ctx, int(variant)), "ac_set_variant")

    def ac_set_upwind(self, on):
        _check(self._lib.ac_set_upwind(self._ctx, int(bool(on))), "ac_set_upwind")

    def ac_set_forcing_mode(self, mode):
        """0 / "rhs" (default, reading G8) or 1 / "kick" (one impulse u += dt f per step)."""
        mode = {"rhs": 0, "kick": 1}.get(mode, mode)
        _check(self._lib.ac_set_forcing_mode(self._ctx, int(mode)), "ac_set_forcing_mode")

    def ac_set_mixed(self, mode):
        """0 / "bidiagonal" (default) or 1 / "tensor"."""
        mode = {"bidiagonal": 0, "tensor": 1}.get(mode, mode)
        _check(self._lib.ac_set_mixed(self._ctx, int(mode)), "ac_set_mixed")

    def ac_launch_count(self):
        return int(self._lib.ac_launch_count(self._ctx))

    def synchronize(self):
        self.stream.synchronize()

    def ac_free(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self._lib.ac_free(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __del__(self):
        try:
            self.ac_free()
        except Exception:
            pass
