"""Thin ctypes binding of include/dmrg.h: argument marshalling only.

Every step of the hot path runs inside libdmrg_b200.so (CUDA, sm_100a).  PyTorch is used by
callers for device memory and streams; this module only converts numpy arrays / tensors to
pointers.  Method names are the C names without the `dmrg_` prefix.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdmrg_b200.so")

OK, EINVAL, ESTATE, ENOMEM, ECUDA, EUNSUPPORTED = 0, -1, -2, -3, -4, -5
SYM_U1U1, SYM_SU2 = 0, 1
PREC_FP64, PREC_FP64_EMU, PREC_TF32X3, PREC_FP64_EMU_PERF = 0, 1, 2, 3
EMU_NO_REF = -(1 << 28)
LEFT_TO_RIGHT, RIGHT_TO_LEFT = 0, 1
(TAB_BOND_L, TAB_BOND_R, TAB_PSI_BLOCKS, TAB_OP_BLOCKS_L, TAB_OP_BLOCKS_R, TAB_GROUPS, TAB_FALG,
 TAB_COUNTS, TAB_ISO_BLOCKS_L, TAB_ISO_BLOCKS_R, TAB_FALG_BLOCKS) = range(11)
OP_I, OP_H, OP_C, OP_S, OP_A, OP_B = range(6)

EXPORTS = [
    "dmrg_create", "dmrg_destroy", "dmrg_last_error", "dmrg_init_integrals", "dmrg_set_mps",
    "dmrg_build_env", "dmrg_plan_bond", "dmrg_psi_length", "dmrg_heff_apply", "dmrg_heff_apply_host",
    "dmrg_heff_diag", "dmrg_davidson_step", "dmrg_renormalize", "dmrg_table", "dmrg_op_export",
    "dmrg_set_timing", "dmrg_last_stage_ms", "dmrg_last_emu_ms", "dmrg_last_emu_stage1_ms", "dmrg_replan", "dmrg_split_truncate", "dmrg_split_result", "dmrg_sweep", "dmrg_measure_peak", "dmrg_emu_gemm", "dmrg_emu_gemm_kept", "dmrg_emu_sum_perf", "dmrg_emu_keep_rule", "dmrg_last_emu_products", "dmrg_launch_count", "dmrg_tf32_split", "dmrg_emu_slice",
    "dmrg_op_export_class", "dmrg_set_option", "dmrg_measure_hbm_kernels", "dmrg_dots", "dmrg_dots_noalloc", "dmrg_noalloc_last_error",
]


class DmrgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"dmrg error {code}: {msg}")
        self.code = code


def load_library(path=None):
    """Load the C-ABI library; fails loudly when it has not been built (no fallback)."""
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(the CUDA library is required; there is no CPU fallback)")
    lib = C.CDLL(path)
    vp, i64p, dp = C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_double)
    lib.dmrg_create.argtypes = [C.POINTER(vp), C.c_int, vp]
    lib.dmrg_destroy.argtypes = [vp]
    lib.dmrg_last_error.argtypes = [vp]
    lib.dmrg_last_error.restype = C.c_char_p
    lib.dmrg_init_integrals.argtypes = [vp, C.c_int, vp, vp, vp, C.c_int, C.c_double, C.c_int, C.c_int,
                                        C.c_int, C.c_int]
    lib.dmrg_set_mps.argtypes = [vp, C.c_int, C.POINTER(vp), i64p, C.POINTER(vp), C.POINTER(vp), i64p,
                                 C.POINTER(vp), C.c_int]
    lib.dmrg_build_env.argtypes = [vp, C.c_int, C.c_int]
    lib.dmrg_plan_bond.argtypes = [vp]
    lib.dmrg_psi_length.argtypes = [vp, i64p]
    lib.dmrg_heff_apply.argtypes = [vp, vp, vp, C.c_int, C.c_int]
    lib.dmrg_heff_apply_host.argtypes = [vp, vp, vp, C.c_int, C.c_int]
    lib.dmrg_heff_diag.argtypes = [vp, vp]
    lib.dmrg_davidson_step.argtypes = [vp, vp, C.c_int, C.c_double, C.c_int, C.c_int, dp, dp,
                                       C.POINTER(C.c_int)]
    lib.dmrg_renormalize.argtypes = [vp, C.c_int, vp, C.c_int64, vp, C.c_int, C.c_int, C.c_int]
    lib.dmrg_table.argtypes = [vp, C.c_int, C.POINTER(i64p), i64p]
    lib.dmrg_op_export.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, vp, C.c_int64]
    lib.dmrg_op_export_class.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, vp, C.c_int64, vp,
                                         C.c_int64, i64p, i64p, i64p]
    lib.dmrg_set_timing.argtypes = [vp, C.c_int]
    lib.dmrg_last_stage_ms.argtypes = [vp, dp, dp]
    lib.dmrg_last_emu_ms.argtypes = [vp, dp, dp]
    lib.dmrg_last_emu_stage1_ms.argtypes = [vp, dp]
    lib.dmrg_replan.argtypes = [vp, C.c_int, C.c_int]
    lib.dmrg_sweep.argtypes = [vp, C.c_int, C.c_int64, C.c_int, C.c_int, C.c_double, C.c_int, C.c_int, C.c_uint64,
                               dp, C.POINTER(C.c_int64), dp]
    lib.dmrg_split_truncate.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int64, dp]
    lib.dmrg_split_result.argtypes = [vp, C.POINTER(C.POINTER(C.c_int64)), C.POINTER(C.c_int64),
                                      C.POINTER(dp), C.POINTER(C.c_int64)]
    lib.dmrg_measure_peak.argtypes = [vp, C.c_int, dp]
    lib.dmrg_emu_gemm.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp, vp, vp, C.c_int, dp, dp]
    lib.dmrg_emu_gemm_kept.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp, vp, vp, C.c_int, C.c_int]
    lib.dmrg_emu_sum_perf.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, vp, vp, vp, vp, C.c_int, C.c_int, vp]
    lib.dmrg_tf32_split.argtypes = [vp, vp, C.c_int64, vp, vp]
    lib.dmrg_emu_keep_rule.argtypes = [vp, vp, vp, C.c_int, C.c_int, C.c_int, vp]
    lib.dmrg_launch_count.argtypes = [vp, C.POINTER(C.c_uint64)]
    lib.dmrg_last_emu_products.argtypes = [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    lib.dmrg_emu_slice.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int64, C.c_int64, C.c_int, vp, vp]
    lib.dmrg_measure_hbm_kernels.argtypes = [vp, vp, C.c_int, dp, dp, C.c_int, C.POINTER(C.c_int)]
    lib.dmrg_set_option.argtypes = [vp, C.c_char_p, C.c_double]
    lib.dmrg_dots.argtypes = [vp, vp, C.c_int64, C.c_int, vp, C.c_int64, vp]
    lib.dmrg_dots_noalloc.argtypes = [vp, vp, C.c_int64, C.c_int, vp, C.c_int64, vp]
    lib.dmrg_noalloc_last_error.argtypes = []
    lib.dmrg_noalloc_last_error.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("dmrg_last_error", "dmrg_noalloc_last_error"):
            getattr(lib, name).restype = C.c_int
    return lib


def _ptr(x):
    """Address of a numpy array, a torch tensor (host or device) or a raw integer."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i64(a):
    return np.ascontiguousarray(a, dtype=np.int64)


class Dmrg:
    """One library context.  device < 0 gives a planning context (tables only, no GPU)."""

    def __init__(self, device=0, stream=None, lib_path=None):
        self.lib = load_library(lib_path)
        self.h = C.c_void_p()
        rc = self.lib.dmrg_create(C.byref(self.h), device, stream)
        if rc != OK:
            raise DmrgError(rc, "dmrg_create failed (no usable sm_100 device; there is no CPU fallback)")
        self._keep = []

    def close(self):
        if self.h:
            self.lib.dmrg_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc):
        if rc != OK:
            raise DmrgError(rc, self.lib.dmrg_last_error(self.h).decode())

    def init_integrals(self, h, V, chol, e_core, N, twoS, symmetry, D):
        h = _f64(h)
        L = h.shape[0]
        V = None if V is None else _f64(V)
        chol = None if chol is None else _f64(chol)
        n_chol = 0 if chol is None else chol.shape[0]
        self._ck(self.lib.dmrg_init_integrals(self.h, L, _ptr(h), _ptr(V), _ptr(chol), n_chol, e_core, N, twoS,
                                              symmetry, D))

    def set_mps(self, bond, left_tables, left_iso, right_tables, right_iso, on_device=False):
        """left_tables[m] (m = 0..bond), left_iso[m] (m = 0..bond-1) packed data; same for the right."""
        def pack(tabs, isos):
            tabs = [_i64(t) for t in tabs]
            tp = (C.c_void_p * len(tabs))(*[t.ctypes.data for t in tabs])
            rows = _i64([t.shape[0] for t in tabs])
            if not on_device:
                isos = [_f64(x) for x in isos]
            ip = (C.c_void_p * max(1, len(isos)))(*[_ptr(x) for x in isos])
            return tabs, tp, rows, isos, ip
        lt, ltp, lrows, li, lip = pack(left_tables, left_iso)
        rt, rtp, rrows, ri, rip = pack(right_tables, right_iso)
        self._ck(self.lib.dmrg_set_mps(self.h, bond, ltp, lrows.ctypes.data_as(C.POINTER(C.c_int64)), lip, rtp,
                                       rrows.ctypes.data_as(C.POINTER(C.c_int64)), rip, int(on_device)))

    def build_env(self, precision=PREC_FP64, slices=0):
        self._ck(self.lib.dmrg_build_env(self.h, precision, slices))

    def plan_bond(self):
        self._ck(self.lib.dmrg_plan_bond(self.h))

    def replan(self, precision=PREC_FP64, slices=0):
        self._ck(self.lib.dmrg_replan(self.h, precision, slices))

    def split_truncate(self, psi, direction, max_states, on_device=True):
        """a10: returns (new bond table [rows, 4], packed isometry, discarded weight)."""
        disc = C.c_double()
        self._ck(self.lib.dmrg_split_truncate(self.h, _ptr(psi), 1 if on_device else 0, direction, max_states, C.byref(disc)))
        tab, iso = C.POINTER(C.c_int64)(), C.POINTER(C.c_double)()
        nt, ni = C.c_int64(), C.c_int64()
        self._ck(self.lib.dmrg_split_result(self.h, C.byref(tab), C.byref(nt), C.byref(iso), C.byref(ni)))
        table = np.ctypeslib.as_array(tab, shape=(nt.value * 4,)).copy().reshape(-1, 4)
        data = np.ctypeslib.as_array(iso, shape=(ni.value,)).copy() if ni.value else np.zeros(0)
        return table, data, disc.value

    def sweep(self, n_sweeps, max_states, davidson_iters=24, max_restarts=12, tol=1e-9, precision=PREC_FP64, slices=0,
              seed=1, L=None):
        """Two-site sweeps on the device; returns (energies of every bond solve, largest discarded weight)."""
        cap = C.c_int64(2 * 4096 * n_sweeps)
        e = np.zeros(cap.value)
        disc = C.c_double()
        self._ck(self.lib.dmrg_sweep(self.h, n_sweeps, max_states, davidson_iters, max_restarts, tol, precision, slices,
                                     seed, e.ctypes.data_as(C.POINTER(C.c_double)), C.byref(cap), C.byref(disc)))
        return e[:cap.value].copy(), disc.value

    def psi_length(self):
        n = C.c_int64()
        self._ck(self.lib.dmrg_psi_length(self.h, C.byref(n)))
        return n.value

    def heff_apply(self, psi_in, psi_out, precision=PREC_FP64, slices=0):
        self._ck(self.lib.dmrg_heff_apply(self.h, _ptr(psi_in), _ptr(psi_out), precision, slices))

    def heff_apply_host(self, psi_in, psi_out, precision=PREC_FP64, slices=0):
        self._ck(self.lib.dmrg_heff_apply_host(self.h, _ptr(psi_in), _ptr(psi_out), precision, slices))

    def heff_diag(self, out):
        self._ck(self.lib.dmrg_heff_diag(self.h, _ptr(out)))

    def davidson_step(self, psi, n_iter, tol=0.0, precision=PREC_FP64, slices=0):
        theta = np.zeros(n_iter)
        resid = np.zeros(n_iter)
        done = C.c_int()
        dp = C.POINTER(C.c_double)
        self._ck(self.lib.dmrg_davidson_step(self.h, _ptr(psi), n_iter, tol, precision, slices,
                                             theta.ctypes.data_as(dp), resid.ctypes.data_as(dp), C.byref(done)))
        return theta[:done.value], resid[:done.value]

    def renormalize(self, direction, new_table, isometry, on_device=False, precision=PREC_FP64, slices=0):
        t = _i64(new_table)
        iso = isometry if on_device else _f64(isometry)
        self._ck(self.lib.dmrg_renormalize(self.h, direction, t.ctypes.data, t.shape[0], _ptr(iso), int(on_device),
                                           precision, slices))

    def table(self, which, ncols=None):
        data = C.POINTER(C.c_int64)()
        n = C.c_int64()
        self._ck(self.lib.dmrg_table(self.h, which, C.byref(data), C.byref(n)))
        a = np.ctypeslib.as_array(data, shape=(n.value,)).copy() if n.value else np.zeros(0, dtype=np.int64)
        return a.reshape(-1, ncols) if ncols else a

    def op_export(self, side, kind, i=-1, k=-1):
        tab = self.table(TAB_BOND_L if side == 0 else TAB_BOND_R, 4)
        dim = int(tab[:, 2].sum())
        out = np.zeros((dim, dim))
        self._ck(self.lib.dmrg_op_export(self.h, side, kind, i, k, out.ctypes.data, dim))
        return out

    def op_export_class(self, side, kind, i0, k0, i_bra, i_ket):
        """Stored blocks <i_bra|O|i_ket> of every operator of one class: (members [n, 2], data [n, rows, cols]);
        (None, None) when the class stores no block for this sector pair."""
        n, r, c = C.c_int64(), C.c_int64(), C.c_int64()
        self._ck(self.lib.dmrg_op_export_class(self.h, side, kind, i0, k0, i_bra, i_ket, None, 0, None, 0,
                                               C.byref(n), C.byref(r), C.byref(c)))
        if n.value == 0:
            return None, None
        out = np.empty((n.value, r.value, c.value))
        mem = np.empty((n.value, 2), dtype=np.int64)
        self._ck(self.lib.dmrg_op_export_class(self.h, side, kind, i0, k0, i_bra, i_ket, out.ctypes.data, out.size,
                                               mem.ctypes.data, n.value, C.byref(n), C.byref(r), C.byref(c)))
        return mem, out

    HBM_NAMES = ["heff_diag", "dots", "ritz_residual", "precondition", "subtract_projection", "slice_psi",
                 "slice_ops_left", "slice_ops_right", "slice_T_unfused"]

    def measure_hbm_kernels(self, psi, n_basis=10):
        """{kernel: {"ms": per launch, "bytes": algorithmic bytes per launch, "GBps": achieved}} (dmrg_measure_hbm_kernels)."""
        ms, by, n = np.zeros(16), np.zeros(16), C.c_int()
        dp = C.POINTER(C.c_double)
        self._ck(self.lib.dmrg_measure_hbm_kernels(self.h, _ptr(psi), n_basis, ms.ctypes.data_as(dp), by.ctypes.data_as(dp), 16,
                                                   C.byref(n)))
        return {name: {"ms": float(ms[i]), "bytes": float(by[i]), "GBps": float(by[i] / (ms[i] * 1e-3) / 1e9)}
                for i, name in enumerate(self.HBM_NAMES[:n.value]) if ms[i] > 0}

    def set_option(self, key, value):
        self._ck(self.lib.dmrg_set_option(self.h, key.encode(), float(value)))

    def dots(self, V, ld, nvec, w, n, out):
        self._ck(self.lib.dmrg_dots(self.h, _ptr(V), ld, nvec, _ptr(w), n, _ptr(out)))

    def set_timing(self, enable=True):
        self._ck(self.lib.dmrg_set_timing(self.h, int(enable)))

    def last_stage_ms(self):
        a, b = C.c_double(), C.c_double()
        self._ck(self.lib.dmrg_last_stage_ms(self.h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def last_emu_ms(self):
        a, b = C.c_double(), C.c_double()
        self._ck(self.lib.dmrg_last_emu_ms(self.h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def last_emu_stage1_ms(self):
        a = C.c_double()
        self._ck(self.lib.dmrg_last_emu_stage1_ms(self.h, C.byref(a)))
        return a.value

    def emu_gemm_kept(self, M, N, K, A, B, Cout, slices, keep):
        self._ck(self.lib.dmrg_emu_gemm_kept(self.h, M, N, K, _ptr(A), _ptr(B), _ptr(Cout), slices, keep))

    def emu_sum_perf(self, M, N, K, A, B, alpha, Cout, slices=0, kmin=3):
        """A: device [n][M][K], B: device [n][K][N]; returns the slice counts the device chose."""
        al = np.ascontiguousarray(alpha, dtype=np.float64)
        keep = np.zeros(len(al), dtype=np.int32)
        self._ck(self.lib.dmrg_emu_sum_perf(self.h, M, N, K, len(al), _ptr(A), _ptr(B), al.ctypes.data, _ptr(Cout), slices, kmin,
                                            keep.ctypes.data))
        return keep.tolist()

    def tf32_split(self, src, n, hi, lo):
        """src: device float64[n]; hi, lo: device int32/uint32[n] receiving FP32 bit patterns."""
        self._ck(self.lib.dmrg_tf32_split(self.h, _ptr(src), n, _ptr(hi), _ptr(lo)))

    def emu_keep_rule(self, E_all, E_nz, slices=0, kmin=3):
        """E_nz entries may be None (no line with a non-zero exponent)."""
        a = np.ascontiguousarray(E_all, dtype=np.int32)
        z = np.ascontiguousarray([EMU_NO_REF if e is None else e for e in E_nz], dtype=np.int32)
        out = np.zeros(len(a), dtype=np.int32)
        self._ck(self.lib.dmrg_emu_keep_rule(self.h, a.ctypes.data, z.ctypes.data, len(a), slices, kmin, out.ctypes.data))
        return out.tolist()

    def launch_count(self):
        n = C.c_uint64(0)
        self._ck(self.lib.dmrg_launch_count(self.h, C.byref(n)))
        return n.value

    def last_emu_products(self):
        a, b = C.c_uint64(0), C.c_uint64(0)
        self._ck(self.lib.dmrg_last_emu_products(self.h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def emu_gemm(self, M, N, K, A, B, Cout, slices=0):
        a, b = C.c_double(), C.c_double()
        self._ck(self.lib.dmrg_emu_gemm(self.h, M, N, K, _ptr(A), _ptr(B), _ptr(Cout), slices, C.byref(a), C.byref(b)))
        return a.value, b.value

    def emu_slice(self, src, lines, K, line_stride, k_stride, slices, out, expo):
        self._ck(self.lib.dmrg_emu_slice(self.h, _ptr(src), lines, K, line_stride, k_stride, slices, _ptr(out),
                                         _ptr(expo)))

    def measure_peak(self, which=PREC_FP64):
        v = C.c_double()
        self._ck(self.lib.dmrg_measure_peak(self.h, which, C.byref(v)))
        return v.value


def dots_noalloc(V, ld, nvec, w, n, out, stream=None, lib=None):
    """dmrg_dots_noalloc: context-free, allocation-free dot products on the current device (see include/dmrg.h)."""
    lib = lib or load_library()
    rc = lib.dmrg_dots_noalloc(stream, _ptr(V), ld, nvec, _ptr(w), n, _ptr(out))
    if rc != OK:
        raise DmrgError(rc, lib.dmrg_noalloc_last_error().decode())
