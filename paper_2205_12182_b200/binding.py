"""ctypes binding of include/nolsm.h. Argument marshalling only: every step of the path runs in the
CUDA kernels behind the C ABI. Arrays may be torch tensors (CPU or CUDA) or numpy arrays."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

PREC_FP16_FP32, PREC_FP32 = 0, 1
DTYPE_F64, DTYPE_F32 = 0, 1
GEMM_AUTO, GEMM_UMMA, GEMM_SIMT = 0, 1, 2
ENGINE_AUTO, ENGINE_PERSISTENT, ENGINE_ROUNDS = 0, 1, 2
ITER_EQ6, ITER_LOWDIN = 0, 1
STATUS_NAMES = {0: "OK", 1: "EINVAL", 2: "ECUDA", 3: "ENOMEM", 4: "ESTATE", 5: "ENOTSPD", 6: "ENOCONV"}

ABI_VERSION = 6                                     # NOLSM_ABI_VERSION of the include/nolsm.h this file restates
_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


class NolsmOptions(C.Structure):
    _fields_ = [("precision", C.c_int), ("gemm_backend", C.c_int), ("max_inv_iters", C.c_int),
                ("max_sign_iters", C.c_int), ("tol_inv", C.c_float), ("tol_sign", C.c_float),
                ("power_iters_s", C.c_int), ("power_iters_a", C.c_int), ("eps_filter", C.c_double),
                ("batch_atoms", C.c_int), ("workspace_bytes", C.c_size_t), ("profile_every", C.c_int),
                ("engine", C.c_int), ("sign_scaled_iters", C.c_int), ("sign_scale", C.c_float),
                ("combine", C.c_int), ("combine_max_dim", C.c_int),
                ("combine_max_members", C.c_int), ("combine_max_candidates", C.c_int), ("iteration", C.c_int),
                ("symmetric_tiles", C.c_int), ("heavy_slots", C.c_int), ("mu_trials", C.c_int),
                ("timeout_s", C.c_double), ("transposed_tiles", C.c_int), ("tuning", C.c_int * 8)]


# names of the engine tuning words options.tuning[k] (include/nolsm.h): accepted as keyword options by Nolsm(...)
TUNING_WORDS = {"claim_lead": 0, "scan_order": 1, "l2_load_policy": 2, "l2_store_policy": 3}


class NolsmStats(C.Structure):
    _fields_ = [("n_atoms", C.c_int64), ("n_batches", C.c_int64), ("dim_min", C.c_int64), ("dim_max", C.c_int64),
                ("dim_mean", C.c_double), ("sum_inv_iters", C.c_int64), ("sum_sign_iters", C.c_int64),
                ("gemms_executed", C.c_int64), ("flops_useful", C.c_double), ("flops_padded", C.c_double),
                ("n_notspd", C.c_int64), ("n_noconv", C.c_int64), ("gather_bytes", C.c_double),
                ("scatter_bytes", C.c_double), ("n_units", C.c_int64), ("gemms_symmetric", C.c_int64),
                ("flops_paper", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class NolsmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"nolsm: {STATUS_NAMES.get(code, code)}: {msg}")
        self.code = code


def lib_path() -> str:
    return os.path.join(_HERE, "libnolsm.so")


def _check_abi(lib, path):
    """Refuses a libnolsm.so built from another header: same version number and the library's sizeof of both structs
    must equal this file's ctypes restatement (a stale library would misread every option behind the first changed field)."""
    stale = f"{path} is stale: rebuild it with `python -m paper_2205_12182_b200.build --force`"
    if not hasattr(lib, "nolsm_abi_version"):
        raise ImportError(f"{stale} (it predates nolsm_abi_version)")
    lib.nolsm_abi_version.restype = C.c_int
    lib.nolsm_sizeof_options.restype = C.c_size_t
    lib.nolsm_sizeof_stats.restype = C.c_size_t
    got = (lib.nolsm_abi_version(), lib.nolsm_sizeof_options(), lib.nolsm_sizeof_stats())
    want = (ABI_VERSION, C.sizeof(NolsmOptions), C.sizeof(NolsmStats))
    if got != want:
        raise ImportError(f"{stale} (ABI version, sizeof(nolsm_options), sizeof(nolsm_stats): library {got}, binding {want})")


def load_library():
    """Loads libnolsm.so (built in-tree by paper_2205_12182_b200/build.py). Fails loudly if absent."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = lib_path()
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -m paper_2205_12182_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(path)
    _check_abi(lib, path)
    P, I64, I32 = C.c_void_p, C.c_int64, C.c_int
    lib.nolsm_create.argtypes = [C.POINTER(P), I32, C.POINTER(NolsmOptions)]
    lib.nolsm_assemble.argtypes = [P, I64, P, P, P, P, P, I32, P]
    lib.nolsm_density_matrix.argtypes = [P, C.c_double, P, I32, P]
    lib.nolsm_density_matrix_range.argtypes = [P, C.c_double, I64, I64, P, I32, C.POINTER(C.c_double), P]
    lib.nolsm_energy.argtypes = [P, C.POINTER(C.c_double)]
    lib.nolsm_destroy.argtypes = [P]
    lib.nolsm_get_index_set.argtypes = [P, I64, P, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    lib.nolsm_electron_count.argtypes = [P, C.POINTER(C.c_double), P]
    lib.nolsm_find_mu.argtypes = [P, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double, I32, P, I32, P,
                                  C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int)]
    lib.nolsm_get_group.argtypes = [P, I64, P, C.POINTER(C.c_int32), P, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    lib.nolsm_gather_submatrix.argtypes = [P, I64, I32, I32, P]
    lib.nolsm_gather_submatrix_noalloc.argtypes = [P, I64, I32, P, P]
    lib.nolsm_get_stats.argtypes = [P, C.POINTER(NolsmStats)]
    lib.nolsm_get_atom_stats.argtypes = [P, I64, I64, P, P, P, P, P, P, P]
    lib.nolsm_get_profile.argtypes = [P, C.POINTER(C.c_double), I32]
    lib.nolsm_get_engine_counters.argtypes = [P, C.POINTER(C.c_double), I32]
    lib.nolsm_electron_counts.argtypes = [P, P, I32, P, P, P]
    lib.nolsm_set_perf_table.argtypes = [P, P, P, I32]
    lib.nolsm_side_task_bandwidth.argtypes = [P, I32, I32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.nolsm_last_error.argtypes = [P]
    lib.nolsm_last_error.restype = C.c_char_p
    for f in ("nolsm_create", "nolsm_assemble", "nolsm_density_matrix", "nolsm_density_matrix_range", "nolsm_energy",
              "nolsm_destroy", "nolsm_get_index_set", "nolsm_get_group", "nolsm_electron_count", "nolsm_find_mu", "nolsm_gather_submatrix", "nolsm_gather_submatrix_noalloc", "nolsm_get_stats",
              "nolsm_get_atom_stats", "nolsm_get_profile", "nolsm_get_engine_counters", "nolsm_electron_counts",
              "nolsm_set_perf_table", "nolsm_side_task_bandwidth"):
        getattr(lib, f).restype = C.c_int
    _LIB = lib
    return lib


def _ptr(a, dtype_np=None, dtype_name=None):
    """(address, keepalive) of a contiguous torch tensor or numpy array."""
    if a is None:
        return None, None
    if hasattr(a, "data_ptr"):                       # torch tensor, any device
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        if dtype_name is not None and str(a.dtype) != "torch." + dtype_name:
            raise TypeError(f"expected torch.{dtype_name}, got {a.dtype}")
        return a.data_ptr(), a
    arr = np.ascontiguousarray(a, dtype=dtype_np)
    return arr.ctypes.data, arr


_VAL = {"float64": DTYPE_F64, "float32": DTYPE_F32}


def _val_dtype(a) -> int:
    name = str(a.dtype).replace("torch.", "")
    if name not in _VAL:
        raise TypeError(f"values must be float64 or float32, got {a.dtype}")
    return _VAL[name]


class Nolsm:
    """nolsm_create / assemble / density_matrix / energy / destroy with the names of include/nolsm.h."""

    def __init__(self, device: int = 0, **opts):
        self._lib = load_library()
        self._h = C.c_void_p()
        o = NolsmOptions()
        for k, v in opts.items():
            if k in TUNING_WORDS:
                o.tuning[TUNING_WORDS[k]] = int(v)
                continue
            if not hasattr(o, k) or k == "tuning":
                raise TypeError(f"unknown option {k}")
            setattr(o, k, v)
        rc = self._lib.nolsm_create(C.byref(self._h), device, C.byref(o))
        if rc:
            self._h = C.c_void_p()
            raise NolsmError(rc, "nolsm_create failed (is a CUDA device visible?)")
        self._keep = []
        self.n_atoms = 0

    def _check(self, rc, soft=()):
        if rc and rc not in soft:
            raise NolsmError(rc, self._lib.nolsm_last_error(self._h).decode())
        return rc

    def assemble(self, atom_nb, row_ptr, col_idx, H0_vals, S_vals, stream: int = 0):
        pa, ka = _ptr(atom_nb, np.int32, "int32")
        pr, kr = _ptr(row_ptr, np.int64, "int64")
        pc, kc = _ptr(col_idx, np.int32, "int32")
        ph, kh = _ptr(H0_vals)
        ps, ks = _ptr(S_vals)
        vd = _val_dtype(kh)
        if _val_dtype(ks) != vd:
            raise TypeError("H0_vals and S_vals must share a dtype")
        self.n_atoms = int(ka.shape[0])
        self._keep = [ka, kr, kc, kh, ks]            # device arrays are borrowed by the library
        self._check(self._lib.nolsm_assemble(self._h, self.n_atoms, pa, pr, pc, ph, ps, vd, stream))

    def density_matrix(self, mu: float, D_vals, stream: int = 0):
        pd, kd = _ptr(D_vals)
        self._keep_out = kd
        self._check(self._lib.nolsm_density_matrix(self._h, float(mu), pd, _val_dtype(kd), stream))

    def density_matrix_range(self, mu: float, atom_begin: int, atom_end: int, D_vals, want_energy=False, stream: int = 0):
        pd, kd = _ptr(D_vals)
        self._keep_out = kd
        e = C.c_double()
        rc = self._lib.nolsm_density_matrix_range(self._h, float(mu), atom_begin, atom_end, pd, _val_dtype(kd),
                                                  C.byref(e) if want_energy else None, stream)
        self._check(rc, soft=(5, 6) if want_energy else ())
        return e.value if want_energy else None

    def energy(self, strict: bool = True) -> float:
        e = C.c_double()
        rc = self._lib.nolsm_energy(self._h, C.byref(e))
        self._check(rc, soft=() if strict else (5, 6))
        return e.value

    def electron_count(self, per_atom: bool = False):
        """Tr(D S) of the last density_matrix call (and the per-atom partials q_i of the evaluated range)."""
        n = C.c_double()
        if not per_atom:
            self._check(self._lib.nolsm_electron_count(self._h, C.byref(n), None))
            return n.value
        q = np.zeros(self.n_atoms, dtype=np.float64)
        self._check(self._lib.nolsm_electron_count(self._h, C.byref(n), q.ctypes.data))
        return n.value, q

    def electron_counts(self, mus, with_energy: bool = False, stream: int = 0, strict: bool = True):
        """Tr(D(mu_j) S) for up to 8 trial mu in one pass over the atoms (include/nolsm.h); no D is written."""
        mu = np.ascontiguousarray(mus, dtype=np.float64)
        n = np.zeros(len(mu), dtype=np.float64)
        e = np.zeros(len(mu), dtype=np.float64)
        self._check(self._lib.nolsm_electron_counts(self._h, mu.ctypes.data, len(mu), n.ctypes.data, e.ctypes.data, stream),
                    soft=() if strict else (5, 6))
        return (n, e) if with_energy else n

    def set_perf_table(self, n, tflops):
        """p(n) of Eq. 10: measured multiplication rate (TFLOP/s) at dimensions n (include/nolsm.h)."""
        nn = np.ascontiguousarray(n, dtype=np.int32)
        tt = np.ascontiguousarray(tflops, dtype=np.float64)
        if len(nn) != len(tt):
            raise ValueError("n and tflops must have the same length")
        self._check(self._lib.nolsm_set_perf_table(self._h, nn.ctypes.data, tt.ctypes.data, len(nn)))

    def side_task_bandwidth(self, which: int, reps: int = 3):
        """(ms per launch, algorithmic bytes per launch) of the gather (0) / scatter (1) task launched alone."""
        ms, by = C.c_double(), C.c_double()
        self._check(self._lib.nolsm_side_task_bandwidth(self._h, which, reps, C.byref(ms), C.byref(by)))
        return ms.value, by.value

    def find_mu(self, n_target: float, mu_lo: float, mu_hi: float, D_vals, tol_n: float = 1e-3, tol_mu: float = 1e-6,
                max_evals: int = 0, stream: int = 0):
        """Bisection on mu until Tr(D S) = n_target (include/nolsm.h). Returns (mu, Tr(D S), evaluations)."""
        pd, kd = _ptr(D_vals)
        self._keep_out = kd
        mu, n, ev = C.c_double(), C.c_double(), C.c_int()
        self._check(self._lib.nolsm_find_mu(self._h, n_target, mu_lo, mu_hi, tol_n, tol_mu, max_evals, pd, _val_dtype(kd), stream,
                                            C.byref(mu), C.byref(n), C.byref(ev)), soft=(6,))
        return mu.value, n.value, ev.value

    def index_set(self, atom: int):
        n = C.c_int32(0)
        dim = C.c_int32(0)
        self._check(self._lib.nolsm_get_index_set(self._h, atom, None, C.byref(n), C.byref(dim)))
        out = np.empty(n.value, dtype=np.int32)
        self._check(self._lib.nolsm_get_index_set(self._h, atom, out.ctypes.data, C.byref(n), C.byref(dim)))
        return out, dim.value

    def group(self, atom: int):
        """(members in joining order, union index set, dimension) of the group `atom` belongs to."""
        nm, ns, dim = C.c_int32(0), C.c_int32(0), C.c_int32(0)
        self._check(self._lib.nolsm_get_group(self._h, atom, None, C.byref(nm), None, C.byref(ns), C.byref(dim)))
        mem = np.empty(nm.value, dtype=np.int32)
        st = np.empty(ns.value, dtype=np.int32)
        self._check(self._lib.nolsm_get_group(self._h, atom, mem.ctypes.data, C.byref(nm), st.ctypes.data, C.byref(ns), C.byref(dim)))
        return mem, st, dim.value

    def gather_submatrix(self, atom: int, which: int, fp16: bool):
        _, _, dim = self.group(atom)                 # the submatrix the atom is evaluated on (its own without combine)
        out = np.empty((dim, dim), dtype=np.float16 if fp16 else np.float32)
        self._check(self._lib.nolsm_gather_submatrix(self._h, atom, which, 1 if fp16 else 0, out.ctypes.data))
        return out

    def gather_submatrix_noalloc(self, atom: int, which: int, out, stream: int = 0):
        """nolsm_gather_submatrix_noalloc (include/nolsm.h): the FP16 gather of the submatrix `atom` is evaluated on, with
        the kernel's scratch in the library's static device array, so the library allocates nothing -- for a process whose
        device memory is all spoken for, or that cannot afford the device-wide wait of a cudaMalloc. `out` is the
        caller's own float16 buffer of dim x dim elements (dim from `group(atom)`): a CUDA tensor (asynchronous on
        `stream`) or a host tensor / numpy array (the call waits). Dimensions beyond 2048 raise. This method allocates
        nothing either; it passes addresses through."""
        if hasattr(out, "data_ptr"):
            if str(out.dtype) != "torch.float16" or not out.is_contiguous():
                raise TypeError("out must be a contiguous float16 tensor")
            addr = out.data_ptr()
        else:
            if out.dtype != np.float16 or not out.flags["C_CONTIGUOUS"]:
                raise TypeError("out must be a C-contiguous float16 array")
            addr = out.ctypes.data
        self._check(self._lib.nolsm_gather_submatrix_noalloc(self._h, atom, which, addr, stream))
        return out

    def stats(self) -> dict:
        s = NolsmStats()
        self._check(self._lib.nolsm_get_stats(self._h, C.byref(s)))
        return s.as_dict()

    def atom_stats(self, atom_begin: int = 0, count: int | None = None) -> dict:
        count = self.n_atoms - atom_begin if count is None else count
        d = {k: np.zeros(count, dtype=np.int32) for k in ("dims", "inv_iters", "sign_iters", "status", "gemms")}
        d["residual"] = np.zeros(count, dtype=np.float32)
        d["e_atom"] = np.zeros(count, dtype=np.float64)
        self._check(self._lib.nolsm_get_atom_stats(self._h, atom_begin, count, *[d[k].ctypes.data for k in
                    ("dims", "inv_iters", "sign_iters", "status", "gemms", "residual", "e_atom")]))
        return d

    def profile(self) -> dict:
        out = (C.c_double * 14)()
        self._check(self._lib.nolsm_get_profile(self._h, out, 14))
        keys = ("gather_ms", "gather_launches", "gather_bytes", "gemm_ms", "gemm_launches", "gemm_flops_useful",
                "gemm_flops_padded", "dcols_ms", "dcols_launches", "dcols_bytes", "other_ms", "other_launches",
                "sampled_submatrices", "kernel_launches")
        return dict(zip(keys, list(out)))

    def engine_counters(self) -> dict:
        """Counters of the persistent engine for the last density_matrix call (include/nolsm.h)."""
        out = (C.c_double * 39)()
        self._check(self._lib.nolsm_get_engine_counters(self._h, out, 39))
        v = list(out)
        kinds = ("none", "refill", "gather", "elementwise", "dcols", "wcols", "k6", "k7")
        d = {"persistent": bool(v[0]), "kernel_ms": v[1], "kernel_ms_device_clock": v[2], "tiles": v[3],
             "sched_idle_ms": v[4], "sched_busy_ms": v[5], "overshoots": v[6], "slots": int(v[7]), "pairs": int(v[8])}
        d["mma_wait_record_ms"], d["mma_wait_accumulator_ms"], d["mma_kloop_ms"] = v[33], v[34], v[35]
        d["sched_wait_ring_ms"], d["sched_wait_claim_point_ms"] = v[36], v[37]
        d["power_steps_extra"] = int(v[38])
        d["side"] = {k: {"busy_ms": v[9 + i], "bytes": v[17 + i], "tasks": v[25 + i]} for i, k in enumerate(kinds)
                     if v[25 + i] > 0}
        return d

    def destroy(self):
        if self._h:
            self._lib.nolsm_destroy(self._h)
            self._h = C.c_void_p()
        self._keep = []

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
