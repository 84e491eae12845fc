"""ctypes binding of libhisq.so (include/hisq.h).  Argument marshalling only: every step of the hot
path runs in the library's CUDA kernels.  PyTorch supplies device memory (tensors) and the stream.

There is deliberately no fallback: if the library is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

from . import layout

HISQ_FP32, HISQ_FP64, HISQ_MIXED = 4, 8, 12
HISQ_EVEN, HISQ_ODD = 0, 1
HISQ_MAX_NRHS = 16
HISQ_EINVAL, HISQ_ENOLINKS, HISQ_ENOWORKSPACE, HISQ_ECUDA = -1, -2, -3, -4
HISQ_ENOCONV, HISQ_EBREAKDOWN, HISQ_EIO, HISQ_EPEER, HISQ_ETOOBIG = -5, -6, -7, -8, -9

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("HISQ_LIB", os.path.join(_HERE, "libhisq.so"))

EXPORTS = [
    "hisq_create", "hisq_destroy", "hisq_set_stream", "hisq_workspace_bytes", "hisq_set_workspace",
    "hisq_set_links", "hisq_dslash", "hisq_apply_A", "hisq_solve_M", "hisq_smear_bytes", "hisq_smear", "hisq_nersc_info", "hisq_nersc_read", "hisq_nersc_write", "hisq_cg", "hisq_cg_multishift", "hisq_set_option", "hisq_get_info", "hisq_spinor_pack",
    "hisq_spinor_unpack", "hisq_dslash_host", "hisq_cg_host", "hisq_naik_compressed", "hisq_launch_count",
    "hisq_create_part", "hisq_peer_bytes", "hisq_peer_attach", "hisq_halo_send", "hisq_halo_recv", "hisq_peer_reduce_send", "hisq_peer_reduce_recv", "hisq_dslash_slices", "hisq_dslash_edges", "hisq_halo_bytes", "hisq_halo_pack", "hisq_halo_unpack",
    "hisq_cgp_begin", "hisq_cgp_phase", "hisq_cgp_ptr", "hisq_cgp_status", "hisq_strerror",
    "hisq_last_error", "hisq_debug_dslash_regs", "hisq_debug_tiles",
    "hisq_cfg_info", "hisq_cfg_read", "hisq_cfg_write",
    "hisq_create_part2", "hisq_zhalo_bytes", "hisq_zhalo_pack", "hisq_zhalo_unpack",
    "hisq_norm2_noalloc", "hisq_norm2_noalloc_max_reals",
]

_lib = None


class HisqError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libhisq error {code}: {msg}")
        self.code = code


def load_library() -> ctypes.CDLL:
    """Load libhisq.so (must have been built: `python -m paper_2306_01098_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2306_01098_b200.build` "
                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i, d, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    lib.hisq_create.argtypes = [ctypes.POINTER(vp), i, i, i, i, i]
    lib.hisq_destroy.argtypes = [vp]
    lib.hisq_set_stream.argtypes = [vp, vp]
    lib.hisq_workspace_bytes.argtypes = [vp, i]
    lib.hisq_workspace_bytes.restype = sz
    lib.hisq_set_workspace.argtypes = [vp, vp, sz]
    lib.hisq_set_links.argtypes = [vp, vp, vp]
    lib.hisq_dslash.argtypes = [vp, vp, vp, i, i]
    lib.hisq_dslash_slices.argtypes = [vp, vp, vp, i, i, i, i]
    lib.hisq_dslash_edges.argtypes = [vp, vp, vp, i, i, i]
    lib.hisq_cg.argtypes = [vp, vp, vp, d, d, i]
    lib.hisq_apply_A.argtypes = [vp, vp, vp, d, i]
    lib.hisq_solve_M.argtypes = [vp, vp, vp, vp, vp, d, d, i]
    lib.hisq_nersc_info.argtypes = [ctypes.c_char_p, ctypes.POINTER(i), ctypes.POINTER(i), ctypes.POINTER(i), ctypes.POINTER(d), ctypes.POINTER(d)]
    lib.hisq_nersc_read.argtypes = [ctypes.c_char_p, vp, sz]
    lib.hisq_nersc_write.argtypes = [ctypes.c_char_p, vp, ctypes.POINTER(i), i, d]
    lib.hisq_cfg_info.argtypes = [ctypes.c_char_p, i, ctypes.POINTER(i), ctypes.POINTER(i)]
    lib.hisq_cfg_read.argtypes = [ctypes.c_char_p, i, vp, sz]
    lib.hisq_cfg_write.argtypes = [ctypes.c_char_p, i, vp, ctypes.POINTER(i), i]
    lib.hisq_norm2_noalloc.argtypes = [vp, i, sz, i, vp, vp]
    lib.hisq_norm2_noalloc_max_reals.argtypes = []
    lib.hisq_norm2_noalloc_max_reals.restype = sz
    lib.hisq_smear_bytes.argtypes = [vp]
    lib.hisq_smear_bytes.restype = sz
    lib.hisq_smear.argtypes = [vp, vp, vp, vp, vp, d, d, i]
    lib.hisq_cg_multishift.argtypes = [vp, vp, vp, d, ctypes.POINTER(d), i, d]
    lib.hisq_set_option.argtypes = [vp, ctypes.c_char_p, d]
    lib.hisq_get_info.argtypes = [vp, ctypes.POINTER(i), ctypes.POINTER(i), ctypes.POINTER(d)]
    lib.hisq_spinor_pack.argtypes = [vp, vp, vp, i]
    lib.hisq_spinor_unpack.argtypes = [vp, vp, vp, i]
    lib.hisq_dslash_host.argtypes = [vp, vp, vp, i, i]
    lib.hisq_cg_host.argtypes = [vp, vp, vp, d, d, i]
    lib.hisq_naik_compressed.argtypes = [vp]
    lib.hisq_create_part.argtypes = [ctypes.POINTER(vp), i, i, i, i, i, i, i]
    lib.hisq_create_part2.argtypes = [ctypes.POINTER(vp), i, i, i, i, i, i, i, i]
    lib.hisq_halo_bytes.argtypes = [vp, i]
    lib.hisq_halo_bytes.restype = sz
    lib.hisq_zhalo_bytes.argtypes = [vp, i]
    lib.hisq_zhalo_bytes.restype = sz
    lib.hisq_zhalo_pack.argtypes = [vp, vp, vp, vp, i]
    lib.hisq_zhalo_unpack.argtypes = [vp, vp, vp, vp, i]
    lib.hisq_peer_bytes.argtypes = [vp, i]
    lib.hisq_peer_bytes.restype = sz
    lib.hisq_peer_attach.argtypes = [vp, ctypes.POINTER(vp), i, i]
    lib.hisq_peer_reduce_send.argtypes = [vp, i, i]
    lib.hisq_peer_reduce_recv.argtypes = [vp, i, i]
    lib.hisq_halo_send.argtypes = [vp, vp, i]
    lib.hisq_halo_recv.argtypes = [vp, vp, i]
    lib.hisq_halo_pack.argtypes = [vp, vp, vp, vp, i]
    lib.hisq_halo_unpack.argtypes = [vp, vp, vp, vp, i]
    lib.hisq_cgp_begin.argtypes = [vp, vp, vp, d, i]
    lib.hisq_cgp_phase.argtypes = [vp, i, d]
    lib.hisq_cgp_ptr.argtypes = [vp, i]
    lib.hisq_cgp_ptr.restype = vp
    lib.hisq_cgp_status.argtypes = [vp, ctypes.POINTER(i), ctypes.POINTER(i), ctypes.POINTER(i), ctypes.POINTER(d)]
    lib.hisq_launch_count.argtypes = [vp]
    lib.hisq_launch_count.restype = ctypes.c_longlong
    lib.hisq_strerror.argtypes = [i]
    lib.hisq_strerror.restype = ctypes.c_char_p
    lib.hisq_last_error.argtypes = [vp]
    lib.hisq_last_error.restype = ctypes.c_char_p
    lib.hisq_debug_dslash_regs.argtypes = [i, i, i]
    lib.hisq_debug_tiles.argtypes = [vp, i, ctypes.POINTER(i)]
    _lib = lib
    return lib


_PREC = {"fp32": HISQ_FP32, "fp64": HISQ_FP64, "mixed": HISQ_MIXED}


def rank_grid(L: Sequence[int], nranks: int):
    """(nz, nt): how the lattice is cut over nranks ranks (hisq_create_part2; rank = rz + nz * rt).  The cut along t alone
    is preferred (contiguous halos); a z cut is added when Lt / nranks is not an even number >= 4 (C5's Lt = 24 on 8
    ranks: 2 x 4).  Raises ValueError if no admissible grid exists."""
    ok = lambda ext, n: ext % n == 0 and (ext // n) % 2 == 0 and ext // n >= 4
    for nz in range(1, int(nranks) + 1):
        if nranks % nz == 0 and ok(L[3], nranks // nz) and (nz == 1 or ok(L[2], nz)):
            return (nz, int(nranks) // nz)
    raise ValueError(f"no (nz, nt) grid of {nranks} ranks fits the lattice {tuple(L)}: local extents must be even and >= 4")


def _grid_of(part):
    """part = (rank, nranks) [t cut only] or (rank, nz, nt) -> (rank, nz, nt)."""
    return (int(part[0]), 1, int(part[1])) if len(part) == 2 else (int(part[0]), int(part[1]), int(part[2]))


class Hisq:
    """One lattice + precision on one GPU.  Method names mirror the C ABI.

    Fields passed to dslash / cg are torch CUDA tensors in the NATIVE layout [nrhs, 3, Vh] complex
    (complex64 for fp32, complex128 otherwise); `pack` / `unpack` convert from / to the canonical
    [nrhs, Vh, 3].  Links are canonical [4, V, 3, 3] complex (Eq. 5: slot mu*V + eo).
    """

    def __init__(self, L: Sequence[int], prec: str = "fp64", nrhs_max: int = 1, device: Optional[torch.device] = None,
                 part: Optional[tuple] = None):
        """part = (rank, nranks): this context is rank's share of the lattice L partitioned along t (hisq_create_part), or
        part = (rank, nz, nt): cut nz times along z and nt times along t (hisq_create_part2, rank = rz + nz * rt);
        self.L then is the EXTENDED local lattice (Lt/nt + 8 slices, and Lz/nz + 8 planes if nz > 1) that every layout
        refers to."""
        layout.check_extents(L)
        self.part = part
        self.L_global = tuple(int(v) for v in L)
        if part is not None:
            rank, nz, nt = _grid_of(part)
            if L[3] % nt or (L[3] // nt) % 2 or L[3] // nt < 4:
                raise ValueError("Lt / nt must be even and >= 4")
            if nz > 1 and (L[2] % nz or (L[2] // nz) % 2 or L[2] // nz < 4):
                raise ValueError("Lz / nz must be even and >= 4")
            self.grid = (nz, nt)
            L = (L[0], L[1], L[2] // nz + (8 if nz > 1 else 0), L[3] // nt + 8)
        if not torch.cuda.is_available():
            raise RuntimeError("libhisq needs a CUDA device (no CPU fallback)")
        self.lib = load_library()
        self.L = tuple(int(v) for v in L)
        self.V = layout.volume(L)
        self.Vh = self.V // 2
        self.prec = prec
        self.device = torch.device(device if device is not None else "cuda:0")
        self.cdtype = torch.complex64 if prec == "fp32" else torch.complex128
        self.nrhs_max = int(nrhs_max)
        self._h = ctypes.c_void_p()
        with torch.cuda.device(self.device):
            if part is None:
                self._check(self.lib.hisq_create(ctypes.byref(self._h), *self.L, _PREC[prec]))
            else:
                self._check(self.lib.hisq_create_part2(ctypes.byref(self._h), *self.L_global, _PREC[prec], *_grid_of(part)))
            self._check(self.lib.hisq_set_stream(self._h, ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)))
            nbytes = self.lib.hisq_workspace_bytes(self._h, self.nrhs_max)
            if nbytes == 0:
                raise HisqError(-1, "hisq_workspace_bytes rejected the arguments")
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self._check(self.lib.hisq_set_workspace(self._h, ctypes.c_void_p(self.workspace.data_ptr()), nbytes))

    # -- plumbing ---------------------------------------------------------------------------------
    def _check(self, code: int, allow=()):
        if code != 0 and code not in allow:
            msg = self.lib.hisq_strerror(code).decode()
            if code == -4 and self._h:
                msg += ": " + self.lib.hisq_last_error(self._h).decode()
            raise HisqError(code, msg)
        return code

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self.lib.hisq_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def use_current_stream(self):
        self._check(self.lib.hisq_set_stream(self._h, ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)))

    def _ptr(self, t: torch.Tensor, shape=None, dtype=None):
        if not t.is_cuda or not t.is_contiguous():
            raise ValueError("expected a contiguous CUDA tensor")
        if dtype is not None and t.dtype != dtype:
            raise ValueError(f"expected dtype {dtype}, got {t.dtype}")
        if shape is not None and tuple(t.shape) != tuple(shape):
            raise ValueError(f"expected shape {tuple(shape)}, got {tuple(t.shape)}")
        return ctypes.c_void_p(t.data_ptr())

    def new_field(self, nrhs: int, native: bool = True) -> torch.Tensor:
        shape = (nrhs, 3, self.Vh) if native else (nrhs, self.Vh, 3)
        return torch.empty(shape, dtype=self.cdtype, device=self.device)

    # -- the C ABI --------------------------------------------------------------------------------
    def set_option(self, key: str, value: float):
        self._check(self.lib.hisq_set_option(self._h, key.encode(), float(value)))

    def set_links(self, fat: torch.Tensor, naik: torch.Tensor):
        shape = (4, self.V, 3, 3)
        self._check(self.lib.hisq_set_links(self._h, self._ptr(fat, shape, self.cdtype), self._ptr(naik, shape, self.cdtype)))

    def pack(self, canonical: torch.Tensor) -> torch.Tensor:
        n = canonical.shape[0]
        out = self.new_field(n, native=True)
        self._check(self.lib.hisq_spinor_pack(self._h, self._ptr(out), self._ptr(canonical, (n, self.Vh, 3), self.cdtype), n))
        return out

    def unpack(self, native: torch.Tensor) -> torch.Tensor:
        n = native.shape[0]
        out = self.new_field(n, native=False)
        self._check(self.lib.hisq_spinor_unpack(self._h, self._ptr(out), self._ptr(native, (n, 3, self.Vh), self.cdtype), n))
        return out

    def dslash(self, inp: torch.Tensor, parity: int, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        n = inp.shape[0]
        if out is None:
            out = self.new_field(n)
        self._check(self.lib.hisq_dslash(self._h, self._ptr(out, (n, 3, self.Vh), self.cdtype),
                                         self._ptr(inp, (n, 3, self.Vh), self.cdtype), int(parity), n))
        return out

    def dslash_slices(self, inp: torch.Tensor, parity: int, out: torch.Tensor, t_first: int, t_count: int) -> torch.Tensor:
        """hisq_dslash_slices: only the owned time slices [t_first, t_first + t_count) of `out` are written."""
        n = inp.shape[0]
        self._check(self.lib.hisq_dslash_slices(self._h, self._ptr(out, (n, 3, self.Vh), self.cdtype),
                                                self._ptr(inp, (n, 3, self.Vh), self.cdtype), int(parity), n,
                                                int(t_first), int(t_count)))
        return out

    def dslash_edges(self, inp: torch.Tensor, parity: int, out: torch.Tensor, width: int) -> torch.Tensor:
        """hisq_dslash_edges: the first and last `width` owned time slices of `out`, one launch."""
        n = inp.shape[0]
        self._check(self.lib.hisq_dslash_edges(self._h, self._ptr(out, (n, 3, self.Vh), self.cdtype),
                                               self._ptr(inp, (n, 3, self.Vh), self.cdtype), int(parity), n, int(width)))
        return out

    def apply_A(self, inp: torch.Tensor, mass: float, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        n = inp.shape[0]
        if out is None:
            out = self.new_field(n)
        self._check(self.lib.hisq_apply_A(self._h, self._ptr(out, (n, 3, self.Vh), self.cdtype),
                                          self._ptr(inp, (n, 3, self.Vh), self.cdtype), float(mass), n))
        return out

    def cg(self, b: torch.Tensor, mass: float, tol: float, x: Optional[torch.Tensor] = None, strict: bool = True):
        """Returns (x, info) with info = dict(iterations, reliable_updates, true_rel_resid, status)."""
        n = b.shape[0]
        if x is None:
            x = self.new_field(n)
        code = self.lib.hisq_cg(self._h, self._ptr(x, (n, 3, self.Vh), self.cdtype), self._ptr(b, (n, 3, self.Vh), self.cdtype),
                                float(mass), float(tol), n)
        self._check(code, allow=() if strict else (HISQ_ENOCONV, HISQ_EBREAKDOWN))
        return x, self.info(n, code)

    def solve_M(self, b_even: torch.Tensor, b_odd: torch.Tensor, mass: float, tol: float, strict: bool = True):
        """(D + mass) x = b on both parities.  Returns (x_even, x_odd, info); info['true_rel_resid'] is the
        full-lattice ||b - M x|| / ||b|| per right-hand side."""
        n = b_even.shape[0]
        xe, xo = self.new_field(n), self.new_field(n)
        shp = (n, 3, self.Vh)
        code = self.lib.hisq_solve_M(self._h, self._ptr(xe, shp, self.cdtype), self._ptr(xo, shp, self.cdtype),
                                     self._ptr(b_even, shp, self.cdtype), self._ptr(b_odd, shp, self.cdtype),
                                     float(mass), float(tol), n)
        self._check(code, allow=() if strict else (HISQ_ENOCONV, HISQ_EBREAKDOWN))
        return xe, xo, self.info(n, code)

    def smear(self, thin: torch.Tensor, fat_scale: float = 1.0, naik_scale: float = -1.0 / 24.0, fold_phases: bool = True):
        """HISQ smearing of canonical thin links [4, V, 3, 3] -> (fat, naik, W), all canonical, ready for set_links."""
        V = 2 * self.Vh
        shp = (4, V, 3, 3)
        fat, naik = torch.empty_like(thin), torch.empty_like(thin)
        nbytes = self.lib.hisq_smear_bytes(self._h)
        scratch = torch.empty(nbytes // thin.element_size(), dtype=thin.dtype, device=thin.device)
        self._check(self.lib.hisq_smear(self._h, self._ptr(thin, shp, self.cdtype), self._ptr(fat, shp, self.cdtype),
                                        self._ptr(naik, shp, self.cdtype), scratch.data_ptr(), float(fat_scale),
                                        float(naik_scale), int(bool(fold_phases))))
        return fat, naik, scratch[4 * V * 9: 8 * V * 9].view(shp)

    def cg_multishift(self, b: torch.Tensor, mass: float, shifts, tol: float, x: Optional[torch.Tensor] = None,
                      strict: bool = True):
        """(mass^2 + shifts[k] - D_eo D_oe) x_k = b; b: [1, 3, Vh]; returns (x [nshift, 3, Vh], info)."""
        ns = len(shifts)
        if x is None:
            x = self.new_field(ns)
        arr = (ctypes.c_double * ns)(*[float(v) for v in shifts])
        code = self.lib.hisq_cg_multishift(self._h, self._ptr(x, (ns, 3, self.Vh), self.cdtype),
                                           self._ptr(b, (1, 3, self.Vh), self.cdtype), float(mass), arr, ns, float(tol))
        self._check(code, allow=() if strict else (HISQ_ENOCONV, HISQ_EBREAKDOWN))
        return x, self.info(ns, code)

    def info(self, nrhs: int, status: int = 0) -> dict:
        it, rel = ctypes.c_int(0), ctypes.c_int(0)
        res = (ctypes.c_double * HISQ_MAX_NRHS)()
        self._check(self.lib.hisq_get_info(self._h, ctypes.byref(it), ctypes.byref(rel), res))
        return {"iterations": it.value, "reliable_updates": rel.value, "true_rel_resid": [res[k] for k in range(nrhs)],
                "status": status}

    # host-buffer (end-to-end) entry points: canonical layout, CPU tensors (pinned or not)
    def dslash_host(self, out_host: torch.Tensor, in_host: torch.Tensor, parity: int):
        n = in_host.shape[0]
        for t in (out_host, in_host):
            if t.is_cuda or not t.is_contiguous() or t.dtype != self.cdtype or tuple(t.shape) != (n, self.Vh, 3):
                raise ValueError("expected contiguous CPU tensors [nrhs, Vh, 3]")
        self._check(self.lib.hisq_dslash_host(self._h, ctypes.c_void_p(out_host.data_ptr()), ctypes.c_void_p(in_host.data_ptr()),
                                              int(parity), n))
        return out_host

    def cg_host(self, x_host: torch.Tensor, b_host: torch.Tensor, mass: float, tol: float, strict: bool = True):
        n = b_host.shape[0]
        for t in (x_host, b_host):
            if t.is_cuda or not t.is_contiguous() or t.dtype != self.cdtype or tuple(t.shape) != (n, self.Vh, 3):
                raise ValueError("expected contiguous CPU tensors [nrhs, Vh, 3]")
        code = self.lib.hisq_cg_host(self._h, ctypes.c_void_p(x_host.data_ptr()), ctypes.c_void_p(b_host.data_ptr()),
                                     float(mass), float(tol), n)
        self._check(code, allow=() if strict else (HISQ_ENOCONV, HISQ_EBREAKDOWN))
        return x_host, self.info(n, code)

    # -- t-partitioned lattices (row f3) -----------------------------------------------------------
    def halo_buffers(self, nrhs: int):
        nb = self.lib.hisq_halo_bytes(self._h, nrhs)
        if nb == 0:
            raise HisqError(-1, "not a partitioned context")
        S = self.Vh // self.L[3]
        mk = lambda: torch.empty((nrhs, 3, 3 * S), dtype=self.cdtype, device=self.device)
        return mk(), mk()

    def halo_pack(self, field: torch.Tensor, lo: torch.Tensor, hi: torch.Tensor):
        self._check(self.lib.hisq_halo_pack(self._h, self._ptr(lo), self._ptr(hi), self._ptr(field), field.shape[0]))

    def halo_unpack(self, field: torch.Tensor, lo: torch.Tensor, hi: torch.Tensor):
        self._check(self.lib.hisq_halo_unpack(self._h, self._ptr(field), self._ptr(lo), self._ptr(hi), field.shape[0]))

    # the same for the z cut (contexts created with nz > 1): 3 planes on each side, owned time slices only
    def zhalo_buffers(self, nrhs: int):
        nb = self.lib.hisq_zhalo_bytes(self._h, nrhs)
        if nb == 0:
            raise HisqError(-1, "not a z-partitioned context")
        n = nb // (nrhs * 3 * (8 if self.prec == "fp32" else 16))
        mk = lambda: torch.empty((nrhs, 3, n), dtype=self.cdtype, device=self.device)
        return mk(), mk()

    def zhalo_pack(self, field: torch.Tensor, lo: torch.Tensor, hi: torch.Tensor):
        self._check(self.lib.hisq_zhalo_pack(self._h, self._ptr(lo), self._ptr(hi), self._ptr(field), field.shape[0]))

    def zhalo_unpack(self, field: torch.Tensor, lo: torch.Tensor, hi: torch.Tensor):
        self._check(self.lib.hisq_zhalo_unpack(self._h, self._ptr(field), self._ptr(lo), self._ptr(hi), field.shape[0]))

    # -- halo transport through peer-mapped mailboxes ------------------------------------------------
    def peer_mailbox(self, nrhs: int) -> torch.Tensor:
        """A zeroed mailbox of hisq_peer_bytes (uint8 device tensor) for this rank; share it with the neighbours."""
        nb = self.lib.hisq_peer_bytes(self._h, nrhs)
        if nb == 0:
            raise HisqError(-1, "not a partitioned context")
        return torch.zeros(nb, dtype=torch.uint8, device=self.device)

    def peer_attach(self, boxes, nrhs: int):
        """boxes[r]: rank r's mailbox as a tensor addressable from this device (own rank: this context's)."""
        self._mailboxes = list(boxes)          # keep the mappings alive as long as the context uses them
        arr = (ctypes.c_void_p * len(boxes))(*[b.data_ptr() for b in boxes])
        self._check(self.lib.hisq_peer_attach(self._h, arr, len(boxes), int(nrhs)))

    def peer_reduce_send(self, which: int, nrhs: int):
        self._check(self.lib.hisq_peer_reduce_send(self._h, int(which), int(nrhs)))

    def peer_reduce_recv(self, which: int, nrhs: int):
        self._check(self.lib.hisq_peer_reduce_recv(self._h, int(which), int(nrhs)))

    def halo_send(self, field: torch.Tensor):
        self._check(self.lib.hisq_halo_send(self._h, self._ptr(field), field.shape[0]))

    def halo_recv(self, field: torch.Tensor):
        self._check(self.lib.hisq_halo_recv(self._h, self._ptr(field), field.shape[0]))

    # -- phase-wise CG (partitioned lattices) ------------------------------------------------------
    def cgp_begin(self, x: torch.Tensor, b: torch.Tensor, tol: float):
        n = b.shape[0]
        self._check(self.lib.hisq_cgp_begin(self._h, self._ptr(x, (n, 3, self.Vh), self.cdtype),
                                            self._ptr(b, (n, 3, self.Vh), self.cdtype), float(tol), n))

    def cgp_phase(self, phase: int, mass: float):
        self._check(self.lib.hisq_cgp_phase(self._h, int(phase), float(mass)))

    def cgp_tensor(self, which: int, nrhs: int) -> torch.Tensor:
        """A torch view (no copy) of library-owned device memory: 0/1 = the p / t field [nrhs, 3, Vh]; 2/3/4 = rho / pq /
        sums [nrhs] float64 -- what the caller exchanges / all-reduces between phases."""
        ptr = self.lib.hisq_cgp_ptr(self._h, int(which))
        if not ptr:
            raise HisqError(-1, "hisq_cgp_ptr")
        base = ptr - self.workspace.data_ptr()
        if which in (0, 1):
            nbytes = nrhs * 3 * self.Vh * (8 if self.prec == "fp32" else 16)
            return self.workspace[base:base + nbytes].view(self.cdtype).view(nrhs, 3, self.Vh)
        return self.workspace[base:base + 8 * nrhs].view(torch.float64)

    def cgp_status(self, nrhs: int) -> dict:
        it, dn, br = ctypes.c_int(0), ctypes.c_int(0), ctypes.c_int(0)
        res = (ctypes.c_double * HISQ_MAX_NRHS)()
        self._check(self.lib.hisq_cgp_status(self._h, ctypes.byref(it), ctypes.byref(dn), ctypes.byref(br), res))
        return {"iterations": it.value, "done": bool(dn.value), "breakdown": bool(br.value),
                "rel_resid": [res[k] for k in range(nrhs)]}

    def naik_compressed(self) -> bool:
        return bool(self.lib.hisq_naik_compressed(self._h))

    def launch_count(self) -> int:
        return int(self.lib.hisq_launch_count(self._h))

    def tiles(self, nrhs: int):
        out = (ctypes.c_int * 2)()
        self._check(self.lib.hisq_debug_tiles(self._h, nrhs, out))
        return out[0], out[1]


# ---- seeded inputs in the layouts the C ABI takes (wraps inputs.py + layout.py; no method arithmetic) -----
def make_links(L, seed: int, device, cdtype=torch.complex128, gen_device=None):
    """(fat, naik) canonical [4, V, 3, 3] on `device`, generated on `gen_device` (default: CPU so the
    numbers are bit-identical to what the oracle's tests see)."""
    from . import inputs
    gdev = torch.device(gen_device) if gen_device is not None else torch.device("cpu")
    sites = layout.lex_of_eo(L, device=gdev)
    fat = inputs.fat_links(L, seed, sites).permute(1, 0, 2, 3).to(cdtype).contiguous().to(device)
    naik = inputs.naik_links(L, seed, sites).permute(1, 0, 2, 3).to(cdtype).contiguous().to(device)
    return fat, naik


def nersc_info(path: str) -> dict:
    """Header of a NERSC-format configuration: L, rows (2 | 3), real_bytes, link_trace, plaquette."""
    lib = load_library()
    L = (ctypes.c_int * 4)()
    rows, rb = ctypes.c_int(0), ctypes.c_int(0)
    lt, pl = ctypes.c_double(0), ctypes.c_double(0)
    code = lib.hisq_nersc_info(path.encode(), L, ctypes.byref(rows), ctypes.byref(rb), ctypes.byref(lt), ctypes.byref(pl))
    if code:
        raise HisqError(code, lib.hisq_strerror(code).decode())
    return {"L": tuple(L), "rows": rows.value, "real_bytes": rb.value, "link_trace": lt.value, "plaquette": pl.value}


def nersc_read(path: str) -> torch.Tensor:
    """A NERSC-format configuration as canonical thin links [4, V, 3, 3] complex128 on the HOST (checksum and link
    trace verified by the library)."""
    lib = load_library()
    L = nersc_info(path)["L"]
    V = L[0] * L[1] * L[2] * L[3]
    out = torch.empty((4, V, 3, 3), dtype=torch.complex128)
    code = lib.hisq_nersc_read(path.encode(), ctypes.c_void_p(out.data_ptr()), out.numel() * 16)
    if code:
        raise HisqError(code, lib.hisq_strerror(code).decode())
    return out


def nersc_write(path: str, links: torch.Tensor, L, rows: int = 3, plaquette: float = 0.0) -> None:
    """Canonical links [4, V, 3, 3] complex128 (host) -> NERSC file (IEEE64BIG)."""
    lib = load_library()
    links = links.to(torch.complex128).cpu().contiguous()
    code = lib.hisq_nersc_write(path.encode(), ctypes.c_void_p(links.data_ptr()), (ctypes.c_int * 4)(*[int(v) for v in L]), int(rows),
                                float(plaquette))
    if code:
        raise HisqError(code, lib.hisq_strerror(code).decode())


def norm2_noalloc(field: torch.Tensor, out: torch.Tensor) -> torch.Tensor:
    """hisq_norm2_noalloc: out[k] = ||field[k]||^2 for a contiguous CUDA tensor field [nrhs, ...] (complex64 / complex128 /
    float32 / float64) into the caller's CUDA tensor `out` (nrhs float64), on the current stream.  The library call
    allocates nothing (static device scratch; at most 16 right-hand sides of 67 108 864 reals: HisqError -9 beyond);
    calls that overlap on the GPU race (include/hisq.h)."""
    lib = load_library()
    if not field.is_cuda or not field.is_contiguous() or not out.is_cuda or not out.is_contiguous():
        raise ValueError("expected contiguous CUDA tensors")
    nrhs = field.shape[0]
    if out.dtype != torch.float64 or out.numel() < nrhs or out.device != field.device:
        raise ValueError("out: float64 CUDA tensor of at least nrhs elements on the field's device")
    real = torch.view_as_real(field) if field.is_complex() else field
    prec = {torch.float32: HISQ_FP32, torch.float64: HISQ_FP64}[real.dtype]
    with torch.cuda.device(field.device):
        code = lib.hisq_norm2_noalloc(ctypes.c_void_p(real.data_ptr()), prec, real.numel() // nrhs, nrhs,
                                      ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
    if code:
        raise HisqError(code, lib.hisq_strerror(code).decode())
    return out


CFG_FORMATS = {"ildg": 1, "milc": 2, "openqcd": 3}


def cfg_info(path: str, fmt: str) -> dict:
    """Header of an ILDG / MILC v5 / openQCD configuration: L = (Lx, Ly, Lz, Lt), real_bytes."""
    lib = load_library()
    L = (ctypes.c_int * 4)()
    rb = ctypes.c_int(0)
    code = lib.hisq_cfg_info(path.encode(), CFG_FORMATS[fmt], L, ctypes.byref(rb))
    if code:
        raise HisqError(code, lib.hisq_strerror(code).decode())
    return {"L": tuple(L), "real_bytes": rb.value}


def cfg_read(path: str, fmt: str) -> torch.Tensor:
    """An ILDG / MILC v5 / openQCD configuration as canonical thin links [4, V, 3, 3] complex128 on the HOST (the
    format's integrity check is verified by the library)."""
    lib = load_library()
    L = cfg_info(path, fmt)["L"]
    V = L[0] * L[1] * L[2] * L[3]
    out = torch.empty((4, V, 3, 3), dtype=torch.complex128)
    code = lib.hisq_cfg_read(path.encode(), CFG_FORMATS[fmt], ctypes.c_void_p(out.data_ptr()), out.numel() * 16)
    if code:
        raise HisqError(code, lib.hisq_strerror(code).decode())
    return out


def cfg_write(path: str, fmt: str, links: torch.Tensor, L, real_bytes: int = 8) -> None:
    """Canonical links [4, V, 3, 3] (host) -> file in the given format."""
    lib = load_library()
    links = links.to(torch.complex128).cpu().contiguous()
    code = lib.hisq_cfg_write(path.encode(), CFG_FORMATS[fmt], ctypes.c_void_p(links.data_ptr()),
                              (ctypes.c_int * 4)(*[int(v) for v in L]), int(real_bytes))
    if code:
        raise HisqError(code, lib.hisq_strerror(code).decode())


def make_thin_links(L, seed: int, device, cdtype=torch.complex128, spread: float = 0.0, gen_device=None):
    """Thin SU(3) links, canonical [4, V, 3, 3] (inputs.thin_links)."""
    from . import inputs
    gdev = torch.device(gen_device) if gen_device is not None else torch.device("cpu")
    sites = layout.lex_of_eo(L, device=gdev)
    return inputs.thin_links(L, seed, sites, spread).permute(1, 0, 2, 3).to(cdtype).contiguous().to(device)


def make_sources(L, seed: int, nrhs: int, parity: int, device, cdtype=torch.complex128, gen_device=None):
    """Gaussian sources on one parity, canonical [nrhs, Vh, 3]."""
    from . import inputs
    gdev = torch.device(gen_device) if gen_device is not None else torch.device("cpu")
    Vh = layout.volume(L) // 2
    sites = layout.lex_of_eo(L, device=gdev)[parity * Vh:(parity + 1) * Vh]
    return inputs.sources(L, seed, sites, nrhs).to(cdtype).contiguous().to(device)
