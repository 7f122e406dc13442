"""ctypes binding of libfourphonon_b200.so -- argument marshalling only (include/fourphonon.h is the contract).

Names follow the C ABI: Context.rates3 -> fp_rates3, Context.rates4 -> fp_rates4, Context.kappa_rta -> fp_kappa_rta,
Context.list3/list4 -> fp_list3/fp_list4.  Arrays may be numpy arrays (HOST entry points: the library does the
host<->device copies itself, inside the call) or torch CUDA tensors (DEVICE entry points).  torch is used only to own
the device workspace and to name the stream.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from dataclasses import dataclass
from pathlib import Path

import numpy as np

FP_OK, FP_EINVAL, FP_ENOMEM, FP_ECUDA, FP_ESTATE = 0, -1, -2, -3, -4
FP_PATH_AUTO, FP_PATH_FUSED, FP_PATH_SPLIT, FP_PATH_SPLIT_SERIAL = 0, 1, 2, 3
FP_PREC_FP64, FP_PREC_MIXED = 0, 1
FP_MEM_HOST, FP_MEM_DEVICE = 0, 1
FP_NOALLOC_MAX_MODES = 65536     # include/fourphonon.h: largest N*nb fp_kappa_rta_static accepts

_PKG = Path(__file__).resolve().parent
_CSRC = _PKG / "csrc"
_LIB = _PKG / "libfourphonon_b200.so"
_SOURCES = ["fp_kernels.cu", "fp_rates.cu", "fp_group.cu", "fp_host.cu", "fp_noalloc.cu"]

# every symbol include/fourphonon.h declares (tests check that the built library exports all of them)
EXPORTED_SYMBOLS = [
    "fp_workspace_bytes", "fp_setup", "fp_rates3", "fp_rates4", "fp_kappa_rta", "fp_kappa_rta_static", "fp_list3", "fp_list4",
    "fp_terms3", "fp_terms4", "fp_set_path", "fp_set_symmetry", "fp_get_symmetry", "fp_set_target_symmetry", "fp_get_target_symmetry", "fp_set_precision", "fp_get_precision", "fp_set_prefilter", "fp_profile_enable", "fp_profile_reset", "fp_profile_get", "fp_probe_fp64_tflops", "fp_probe_dmma_tflops", "fp_constants",
    "fp_last_error", "fp_version", "fp_destroy",
]


class FourPhononError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"fourphonon error {code}: {msg}")
        self.code = code


def library_path() -> Path:
    return _LIB


def build_library(force: bool = False, verbose: bool = False) -> Path:
    """nvcc -gencode arch=compute_100a,code=sm_100a (cross-compiles without a GPU); in-tree so it ships with gpurun."""
    srcs = [_CSRC / s for s in _SOURCES]
    deps = srcs + [_CSRC / "fp_internal.cuh", _CSRC / "fp_device.cuh", _CSRC / "fp_contract.cuh", _PKG.parent / "include" / "fourphonon.h"]
    if not force and _LIB.exists() and all(_LIB.stat().st_mtime >= d.stat().st_mtime for d in deps):
        return _LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-Xcompiler", "-fPIC,-ffp-contract=off", "-shared", "-o", str(_LIB)] + [str(s) for s in srcs]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    extra = os.environ.get("FP_NVCC_EXTRA", "").split()               # tuning experiments: -D knobs of the kernels
    cmd[1:1] = extra
    subprocess.run(cmd, check=True)
    return _LIB


class _Crystal(C.Structure):
    _fields_ = [("lattvec", C.c_double * 9), ("natoms", C.c_int32)]


class _Ifc(C.Structure):
    _fields_ = [("n", C.c_int64), ("atoms", C.c_void_p), ("cells", C.c_void_p), ("phi", C.c_void_p)]


class _Broadening(C.Structure):
    _fields_ = [("scale", C.c_double), ("ncut", C.c_double), ("sigma_const", C.c_double)]


class _Profile(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("ms_precontract", "ms_rates", "ms_reduce")] + \
               [(n, C.c_int64) for n in ("n_precontract", "n_rates", "n_reduce", "rows", "candidates", "prefiltered",
                                         "processes")] + [("rates_flops", C.c_double), ("ms_enum", C.c_double),
                                                          ("n_enum", C.c_int64), ("evaluated", C.c_int64),
                                                          ("list_overflows", C.c_int64)]


@dataclass
class Profile:
    ms_precontract: float
    ms_rates: float
    ms_reduce: float
    n_precontract: int
    n_rates: int
    n_reduce: int
    rows: int
    candidates: int
    prefiltered: int
    processes: int
    rates_flops: float
    ms_enum: float = 0.0
    n_enum: int = 0
    evaluated: int = 0
    list_overflows: int = 0

    @property
    def launches(self) -> int:
        return self.n_precontract + self.n_rates + self.n_reduce + self.n_enum


_lib = None


def load_library():
    """Load the CUDA library; fails loudly if it has not been built (no CPU fallback exists)."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB.exists():
        raise FourPhononError(FP_ESTATE, f"{_LIB} is missing: run __graft_entry__.build() (nvcc, sm_100a) first")
    lib = C.CDLL(str(_LIB))
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.fp_workspace_bytes.restype = C.c_size_t
    lib.fp_workspace_bytes.argtypes = [C.POINTER(_Crystal), C.POINTER(i32), C.POINTER(_Ifc), C.POINTER(_Ifc), C.c_size_t]
    lib.fp_setup.restype = C.c_int
    lib.fp_setup.argtypes = [C.POINTER(_Crystal), vp, vp, vp, vp, C.c_int, C.POINTER(_Ifc), C.POINTER(_Ifc),
                             C.POINTER(i32), dbl, C.POINTER(_Broadening), vp, C.c_size_t, vp, C.POINTER(vp)]
    lib.fp_rates3.restype = C.c_int
    lib.fp_rates3.argtypes = [vp, vp, i64, vp, vp, vp, C.c_int, vp]
    lib.fp_rates4.restype = C.c_int
    lib.fp_rates4.argtypes = [vp, vp, i64, i32, i32, vp, vp, vp, C.c_int, vp]
    lib.fp_kappa_rta.restype = C.c_int
    lib.fp_kappa_rta.argtypes = [vp, vp, vp, C.c_int, vp]
    lib.fp_kappa_rta_static.restype = C.c_int
    lib.fp_kappa_rta_static.argtypes = [vp, vp, vp, C.c_int, vp]
    lib.fp_list3.restype = C.c_int
    lib.fp_list3.argtypes = [vp, i32, i32, vp, i64, C.POINTER(i64), vp]
    lib.fp_list4.restype = C.c_int
    lib.fp_list4.argtypes = [vp, i32, i32, i32, vp, i64, C.POINTER(i64), vp]
    lib.fp_terms3.restype = C.c_int
    lib.fp_terms3.argtypes = [vp, i32, i32, vp, vp, i64, C.POINTER(i64), vp]
    lib.fp_terms4.restype = C.c_int
    lib.fp_terms4.argtypes = [vp, i32, i32, i32, vp, vp, i64, C.POINTER(i64), vp]
    lib.fp_set_path.restype = C.c_int
    lib.fp_set_path.argtypes = [vp, C.c_int]
    lib.fp_set_symmetry.restype = C.c_int
    lib.fp_set_symmetry.argtypes = [vp, C.c_int]
    lib.fp_get_symmetry.restype = C.c_int
    lib.fp_get_symmetry.argtypes = [vp]
    lib.fp_set_target_symmetry.restype = C.c_int
    lib.fp_set_target_symmetry.argtypes = [vp, C.c_int]
    lib.fp_get_target_symmetry.restype = C.c_int
    lib.fp_get_target_symmetry.argtypes = [vp]
    lib.fp_set_precision.restype = C.c_int
    lib.fp_set_precision.argtypes = [vp, C.c_int]
    lib.fp_get_precision.restype = C.c_int
    lib.fp_get_precision.argtypes = [vp]
    lib.fp_set_prefilter.restype = C.c_int
    lib.fp_set_prefilter.argtypes = [vp, C.c_int]
    lib.fp_profile_enable.restype = C.c_int
    lib.fp_profile_enable.argtypes = [vp, C.c_int]
    lib.fp_profile_reset.restype = C.c_int
    lib.fp_profile_reset.argtypes = [vp]
    lib.fp_profile_get.restype = C.c_int
    lib.fp_profile_get.argtypes = [vp, C.POINTER(_Profile)]
    lib.fp_probe_fp64_tflops.restype = C.c_int
    lib.fp_probe_fp64_tflops.argtypes = [vp, C.POINTER(dbl)]
    lib.fp_probe_dmma_tflops.restype = C.c_int
    lib.fp_probe_dmma_tflops.argtypes = [vp, C.POINTER(dbl)]
    lib.fp_constants.restype = None
    lib.fp_constants.argtypes = [C.POINTER(dbl)]
    lib.fp_last_error.restype = C.c_char_p
    lib.fp_last_error.argtypes = [vp]
    lib.fp_version.restype = C.c_char_p
    lib.fp_destroy.restype = C.c_int
    lib.fp_destroy.argtypes = [vp]
    _lib = lib
    return lib


def fp_version() -> str:
    return load_library().fp_version().decode()


def fp_constants() -> dict:
    out = (C.c_double * 4)()
    load_library().fp_constants(out)
    return {"C3": out[0], "C4": out[1], "Ckappa": out[2], "hbar_over_kb": out[3]}


def _stream_ptr(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if hasattr(stream, "cuda_stream"):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


def fp_probe_fp64_tflops(stream=None) -> float:
    out = C.c_double(0.0)
    rc = load_library().fp_probe_fp64_tflops(_stream_ptr(stream), C.byref(out))
    if rc != FP_OK:
        raise FourPhononError(rc, "fp_probe_fp64_tflops failed")
    return out.value


def fp_probe_dmma_tflops(stream=None) -> dict:
    """TFLOP/s of DMMA.8x8x4 alone, DFMA alone and both interleaved (include/fourphonon.h)."""
    out = (C.c_double * 3)()
    rc = load_library().fp_probe_dmma_tflops(_stream_ptr(stream), out)
    if rc != FP_OK:
        raise FourPhononError(rc, "fp_probe_dmma_tflops failed")
    return {"dmma": out[0], "dfma": out[1], "dmma_and_dfma": out[2]}


def _is_torch(x):
    return hasattr(x, "data_ptr") and hasattr(x, "is_cuda")


def _ifc_struct(ifc, order, keep):
    if ifc is None:
        return None
    atoms = np.ascontiguousarray(ifc[0], dtype=np.int32).reshape(-1, order)
    cells = np.ascontiguousarray(ifc[1], dtype=np.int32).reshape(-1, order - 1, 3)
    phi = np.ascontiguousarray(ifc[2], dtype=np.float64).reshape(-1, 3 ** order)
    if not (atoms.shape[0] == cells.shape[0] == phi.shape[0]):
        raise FourPhononError(FP_EINVAL, "IFC arrays disagree on the number of clusters")
    keep += [atoms, cells, phi]
    s = _Ifc()
    s.n = atoms.shape[0]
    s.atoms, s.cells, s.phi = atoms.ctypes.data, cells.ctypes.data, phi.ctypes.data
    return s


class Context:
    """fp_setup ... fp_destroy.  Owns the device workspace (a torch uint8 CUDA tensor) for the context's lifetime."""

    def __init__(self, lattvec, masses, omega, eig, vg, mesh, T=300.0, ifc3=None, ifc4=None, scale=1.0, ncut=2.0,
                 sigma_const=0.0, scratch_bytes=1 << 30, device="cuda:0", stream=None, workspace_bytes=None):
        import torch
        self._torch = torch
        self.lib = load_library()
        self.ctx = C.c_void_p(None)
        self.device = torch.device(device)
        masses = np.ascontiguousarray(masses, dtype=np.float64).reshape(-1)
        natoms = masses.size
        self.nb = 3 * natoms
        self.mesh = np.ascontiguousarray(mesh, dtype=np.int32).reshape(3)
        self.N = int(np.prod(self.mesh.astype(np.int64)))
        self.nmodes = self.N * self.nb
        cr = _Crystal()
        cr.lattvec = (C.c_double * 9)(*[float(x) for x in np.asarray(lattvec, dtype=np.float64).reshape(-1)])
        cr.natoms = natoms
        keep = []
        s3, s4 = _ifc_struct(ifc3, 3, keep), _ifc_struct(ifc4, 4, keep)
        p3 = C.byref(s3) if s3 is not None else None
        p4 = C.byref(s4) if s4 is not None else None
        mesh_c = (C.c_int32 * 3)(*[int(x) for x in self.mesh])
        br = _Broadening(float(scale), float(ncut), float(sigma_const))

        dev_in = _is_torch(omega)
        if dev_in:
            if not (_is_torch(eig) and _is_torch(vg) and omega.is_cuda and eig.is_cuda and vg.is_cuda):
                raise FourPhononError(FP_EINVAL, "omega, eig, vg must all be CUDA tensors or all be numpy arrays")
            omega = omega.contiguous().to(torch.float64)
            eig = eig.contiguous()
            eig = torch.view_as_real(eig) if eig.is_complex() else eig.to(torch.float64)
            eig = eig.contiguous()
            vg = vg.contiguous().to(torch.float64)
            shapes = (omega.numel(), eig.numel(), vg.numel())
            ptrs = (omega.data_ptr(), eig.data_ptr(), vg.data_ptr())
            keep += [omega, eig, vg]
        else:
            omega = np.ascontiguousarray(omega, dtype=np.float64)
            eig = np.ascontiguousarray(eig)
            eig = eig.astype(np.complex128).view(np.float64) if np.iscomplexobj(eig) else eig.astype(np.float64)
            eig = np.ascontiguousarray(eig)
            vg = np.ascontiguousarray(vg, dtype=np.float64)
            shapes = (omega.size, eig.size, vg.size)
            ptrs = (omega.ctypes.data, eig.ctypes.data, vg.ctypes.data)
            keep += [omega, eig, vg]
        if shapes != (self.nmodes, self.nmodes * self.nb * 2, self.nmodes * 3):
            raise FourPhononError(FP_EINVAL, f"mode array sizes {shapes} do not match mesh {self.mesh} x {self.nb} branches")

        nbytes = self.lib.fp_workspace_bytes(C.byref(cr), mesh_c, p3, p4, int(scratch_bytes))
        if nbytes == 0:
            raise FourPhononError(FP_EINVAL, "fp_workspace_bytes rejected the arguments")
        if workspace_bytes is not None:                                # caller-chosen size (fp_setup checks it)
            nbytes = int(workspace_bytes)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            off = (-self.workspace.data_ptr()) % 256
            self._ws_ptr = self.workspace.data_ptr() + off
            rc = self.lib.fp_setup(C.byref(cr), masses.ctypes.data, ptrs[0], ptrs[1], ptrs[2],
                                   FP_MEM_DEVICE if dev_in else FP_MEM_HOST, p3, p4, mesh_c, float(T), C.byref(br),
                                   C.c_void_p(self._ws_ptr), nbytes, _stream_ptr(stream), C.byref(self.ctx))
        if rc != FP_OK:
            msg = self.lib.fp_last_error(None).decode()
            self.ctx = C.c_void_p(None)
            raise FourPhononError(rc, msg)

    # -- helpers ---------------------------------------------------------------------------------------------------------
    def _check(self, rc):
        if rc != FP_OK:
            raise FourPhononError(rc, self.lib.fp_last_error(self.ctx).decode())

    def close(self):
        if getattr(self, "ctx", None) is not None and self.ctx.value:
            self.lib.fp_destroy(self.ctx)
            self.ctx = C.c_void_p(None)
        self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def _rates(self, order, targets, qp_begin, qp_end, stream, out):
        torch = self._torch
        nch = 2 if order == 3 else 3
        if _is_torch(targets):
            t = targets.contiguous().to(torch.int32)
            nt = t.numel()
            if out is None:
                g = torch.empty((nt, nch), dtype=torch.float64, device=t.device)
                w = torch.empty((nt, nch), dtype=torch.float64, device=t.device)
                c = torch.empty((nt, nch), dtype=torch.int64, device=t.device)
            else:
                g, w, c = out
            ptrs = (t.data_ptr(), g.data_ptr(), w.data_ptr(), c.data_ptr())
            loc = FP_MEM_DEVICE
        else:
            t = np.ascontiguousarray(targets, dtype=np.int32).reshape(-1)
            nt = t.size
            if out is None:
                g = np.zeros((nt, nch)); w = np.zeros((nt, nch)); c = np.zeros((nt, nch), dtype=np.int64)
            else:
                g, w, c = out
            ptrs = (t.ctypes.data, g.ctypes.data, w.ctypes.data, c.ctypes.data)
            loc = FP_MEM_HOST
        with torch.cuda.device(self.device):
            if order == 3:
                rc = self.lib.fp_rates3(self.ctx, ptrs[0], nt, ptrs[1], ptrs[2], ptrs[3], loc, _stream_ptr(stream))
            else:
                rc = self.lib.fp_rates4(self.ctx, ptrs[0], nt, int(qp_begin), int(self.N if qp_end is None else qp_end),
                                        ptrs[1], ptrs[2], ptrs[3], loc, _stream_ptr(stream))
        self._check(rc)
        return g, w, c

    # -- the C ABI ---------------------------------------------------------------------------------------------------------
    def rates3(self, targets, stream=None, out=None):
        """fp_rates3: (gamma[nt,2], wp[nt,2], counts[nt,2]) for channels (+,-)."""
        return self._rates(3, targets, 0, 1, stream, out)

    def rates4(self, targets, qp_begin=0, qp_end=None, stream=None, out=None):
        """fp_rates4: (gamma[nt,3], wp[nt,3], counts[nt,3]) for channels (++,+-,--), q' in [qp_begin, qp_end)."""
        return self._rates(4, targets, qp_begin, qp_end, stream, out)

    def kappa_rta(self, gamma_total, stream=None):
        """fp_kappa_rta: 3x3 kappa (W/mK) from total rates [N*nb] (1/ps)."""
        torch = self._torch
        with torch.cuda.device(self.device):
            if _is_torch(gamma_total):
                g = gamma_total.contiguous().to(torch.float64).reshape(-1)
                if g.numel() != self.nmodes:
                    raise FourPhononError(FP_EINVAL, "gamma_total must have N*nb entries")
                k = torch.empty((3, 3), dtype=torch.float64, device=g.device)
                rc = self.lib.fp_kappa_rta(self.ctx, g.data_ptr(), k.data_ptr(), FP_MEM_DEVICE, _stream_ptr(stream))
            else:
                g = np.ascontiguousarray(gamma_total, dtype=np.float64).reshape(-1)
                if g.size != self.nmodes:
                    raise FourPhononError(FP_EINVAL, "gamma_total must have N*nb entries")
                k = np.zeros((3, 3))
                rc = self.lib.fp_kappa_rta(self.ctx, g.ctypes.data, k.ctypes.data, FP_MEM_HOST, _stream_ptr(stream))
        self._check(rc)
        return k

    def kappa_rta_static(self, gamma_total, stream=None):
        """fp_kappa_rta_static: kappa_rta without any allocation on the library side (static device scratch; N*nb <=
        FP_NOALLOC_MAX_MODES; calls that overlap on the GPU race).  numpy in -> numpy out, torch CUDA in -> torch out."""
        torch = self._torch
        with torch.cuda.device(self.device):
            if _is_torch(gamma_total):
                g = gamma_total.contiguous().to(torch.float64).reshape(-1)
                if g.numel() != self.nmodes:
                    raise FourPhononError(FP_EINVAL, "gamma_total must have N*nb entries")
                k = torch.empty((3, 3), dtype=torch.float64, device=g.device)
                rc = self.lib.fp_kappa_rta_static(self.ctx, g.data_ptr(), k.data_ptr(), FP_MEM_DEVICE, _stream_ptr(stream))
            else:
                g = np.ascontiguousarray(gamma_total, dtype=np.float64).reshape(-1)
                if g.size != self.nmodes:
                    raise FourPhononError(FP_EINVAL, "gamma_total must have N*nb entries")
                k = np.zeros((3, 3))
                rc = self.lib.fp_kappa_rta_static(self.ctx, g.ctypes.data, k.ctypes.data, FP_MEM_HOST, _stream_ptr(stream))
        self._check(rc)
        return k

    def list3(self, target, channel, stream=None):
        """fp_list3: allowed (lambda', lambda'') pairs of one target and channel (debug export)."""
        n = C.c_int64(0)
        with self._torch.cuda.device(self.device):
            self._check(self.lib.fp_list3(self.ctx, int(target), int(channel), None, 0, C.byref(n), _stream_ptr(stream)))
            out = np.zeros((max(n.value, 1), 2), dtype=np.int32)
            self._check(self.lib.fp_list3(self.ctx, int(target), int(channel), out.ctypes.data, n.value, C.byref(n),
                                          _stream_ptr(stream)))
        return out[:n.value]

    def list4(self, target, channel, qp, stream=None):
        """fp_list4: allowed (lambda', lambda'', lambda''') triples of one target, channel and q' (debug export)."""
        n = C.c_int64(0)
        with self._torch.cuda.device(self.device):
            self._check(self.lib.fp_list4(self.ctx, int(target), int(channel), int(qp), None, 0, C.byref(n),
                                          _stream_ptr(stream)))
            out = np.zeros((max(n.value, 1), 3), dtype=np.int32)
            self._check(self.lib.fp_list4(self.ctx, int(target), int(channel), int(qp), out.ctypes.data, n.value,
                                          C.byref(n), _stream_ptr(stream)))
        return out[:n.value]

    def terms3(self, target, channel, stream=None):
        """fp_terms3: the 3ph process list of one target and channel and each process's contribution to Gamma."""
        n = C.c_int64(0)
        with self._torch.cuda.device(self.device):
            self._check(self.lib.fp_terms3(self.ctx, int(target), int(channel), None, None, 0, C.byref(n), _stream_ptr(stream)))
            out = np.zeros((max(n.value, 1), 2), dtype=np.int32)
            g = np.zeros(max(n.value, 1), dtype=np.float64)
            self._check(self.lib.fp_terms3(self.ctx, int(target), int(channel), out.ctypes.data, g.ctypes.data, n.value,
                                           C.byref(n), _stream_ptr(stream)))
        return out[:n.value], g[:n.value]

    def terms4(self, target, channel, qp, stream=None):
        """fp_terms4: the 4ph process list of one target, channel and q-prime and each process's contribution to Gamma."""
        n = C.c_int64(0)
        with self._torch.cuda.device(self.device):
            self._check(self.lib.fp_terms4(self.ctx, int(target), int(channel), int(qp), None, None, 0, C.byref(n),
                                           _stream_ptr(stream)))
            out = np.zeros((max(n.value, 1), 3), dtype=np.int32)
            g = np.zeros(max(n.value, 1), dtype=np.float64)
            self._check(self.lib.fp_terms4(self.ctx, int(target), int(channel), int(qp), out.ctypes.data, g.ctypes.data,
                                           n.value, C.byref(n), _stream_ptr(stream)))
        return out[:n.value], g[:n.value]

    def set_path(self, path: int):
        """FP_PATH_AUTO / FP_PATH_FUSED / FP_PATH_SPLIT / FP_PATH_SPLIT_SERIAL (include/fourphonon.h)."""
        self._check(self.lib.fp_set_path(self.ctx, int(path)))

    def set_symmetry(self, on: bool):
        """Turn the lambda'' <-> lambda''' pair reuse of the 4ph +- / -- channels on or off (include/fourphonon.h)."""
        self._check(self.lib.fp_set_symmetry(self.ctx, 1 if on else 0))

    def set_target_symmetry(self, on: bool):
        """fp_set_target_symmetry: time-reversal reuse between the targets (q,j) and (-q,j) of one call."""
        self._check(self.lib.fp_set_target_symmetry(self.ctx, 1 if on else 0))

    def get_target_symmetry(self) -> bool:
        """True if fp_setup found the mode arrays time-reversal symmetric bit for bit and the reuse is on."""
        return self.lib.fp_get_target_symmetry(self.ctx) > 0

    def set_precision(self, mode: int):
        """fp_set_precision: FP_PREC_FP64 (default) or FP_PREC_MIXED (level-2 contraction in FP32; include/fourphonon.h)."""
        self._check(self.lib.fp_set_precision(self.ctx, int(mode)))

    def get_precision(self) -> int:
        return int(self.lib.fp_get_precision(self.ctx))

    def set_prefilter(self, on: bool):
        """fp_set_prefilter: False disables every FP32 pre-filter test (self-check of the superset claim; slow)."""
        self._check(self.lib.fp_set_prefilter(self.ctx, 1 if on else 0))

    def get_symmetry(self) -> bool:
        """True if fp_setup found an IFC list symmetric in its last two legs and the reuse is on (get_symmetry_mask: which)."""
        return self.lib.fp_get_symmetry(self.ctx) > 0

    def get_symmetry_mask(self) -> int:
        """bit 0: 3ph - channel, bit 1: 4ph +- and -- channels"""
        return int(self.lib.fp_get_symmetry(self.ctx))

    def profile_enable(self, on=True):
        self._check(self.lib.fp_profile_enable(self.ctx, 1 if on else 0))

    def profile_reset(self):
        self._check(self.lib.fp_profile_reset(self.ctx))

    def profile_get(self) -> Profile:
        p = _Profile()
        self._check(self.lib.fp_profile_get(self.ctx, C.byref(p)))
        return Profile(**{n: getattr(p, n) for n, _ in _Profile._fields_})

    @classmethod
    def from_inputs(cls, inp, **kw):
        """Convenience for fp_inputs.Inputs (host arrays)."""
        kw.setdefault("T", inp.T)
        kw.setdefault("scale", inp.scale)
        return cls(inp.crystal.lattvec, inp.crystal.masses, inp.omega, inp.eig, inp.vg, inp.mesh, ifc3=inp.ifc3,
                   ifc4=inp.ifc4, **kw)
