"""Thin ctypes binding of include/frb200.h -- argument marshalling only; every step of the hot path runs in
the CUDA kernels of libfrb200.so.  PyTorch is used by callers for device memory and streams only.
There is no CPU fallback: a missing library or a missing GPU raises."""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfrb200.so")

FR_OK, FR_EINVAL, FR_ENOMEM, FR_ECUDA, FR_ESTATE, FR_EUNSUPPORTED = range(6)
FR_F32, FR_F64 = 4, 8
FR_EULER, FR_NAVIER_STOKES = 0, 1
FR_TET, FR_PRI, FR_HEX = 0, 1, 2
FR_RK4, FR_RK45_2R, FR_EULER1 = 0, 1, 2
FR_BC_NOSLIP_ISOTHERMAL_WALL, FR_BC_CHAR_RIEMANN_INV = 0, 1
FR_MODE_FUSED, FR_MODE_UNFUSED = 0, 1

_dp = C.POINTER(C.c_double)
_i32p = C.POINTER(C.c_int32)
_i64p = C.POINTER(C.c_int64)


class fr_eles_desc(C.Structure):
    _fields_ = [("etype", C.c_int), ("order", C.c_int32), ("nupts", C.c_int32), ("nfpts", C.c_int32),
                ("neles", C.c_int64), ("affine", C.c_int32),
                ("M0", _dp), ("M132", _dp), ("M3", _dp), ("M460", _dp), ("M6", _dp), ("smats", _dp), ("rcpdjac", _dp)]


class fr_iface_desc(C.Structure):
    _fields_ = [("npairs", C.c_int64), ("l_et", _i32p), ("l_fpt", _i32p), ("l_ele", _i64p),
                ("r_et", _i32p), ("r_fpt", _i32p), ("r_ele", _i64p), ("nl", _dp), ("magl", _dp), ("magr", _dp)]


class fr_bc_desc(C.Structure):
    _fields_ = [("type", C.c_int), ("nfpts", C.c_int64), ("et", _i32p), ("fpt", _i32p), ("ele", _i64p),
                ("n", _dp), ("mag", _dp), ("params", C.c_double * 8)]


class fr_halo_desc(C.Structure):
    _fields_ = [("nghost", C.c_int64), ("et", _i32p), ("fpt", _i32p), ("ele", _i64p)]


class fr_config(C.Structure):
    _fields_ = [("system", C.c_int), ("prec", C.c_int), ("stepper", C.c_int), ("mode", C.c_int),
                ("gamma", C.c_double), ("mu", C.c_double), ("prandtl", C.c_double),
                ("ldg_beta", C.c_double), ("ldg_tau", C.c_double),
                ("netypes", C.c_int32), ("eles", C.POINTER(fr_eles_desc)), ("ifaces", C.POINTER(fr_iface_desc)),
                ("nbcs", C.c_int32), ("bcs", C.POINTER(fr_bc_desc)), ("cuda_stream", C.c_void_p),
                ("halo", C.POINTER(fr_halo_desc))]


class fr_kernel_stat(C.Structure):
    _fields_ = [("name", C.c_char * 48), ("ms", C.c_double), ("alg_bytes", C.c_double), ("flops", C.c_double),
                ("category", C.c_int32)]


class fr_adapt_stats(C.Structure):
    _fields_ = [("accepted", C.c_int64), ("rejected", C.c_int64), ("t", C.c_double), ("dt_next", C.c_double)]


GEMM_STATIC_MAX_BYTES = 512 * 1024     # FR_GEMM_STATIC_MAX_BYTES of include/frb200.h

SYMBOLS = ["fr_profile_kernels", "fr_rk_step_host", "fr_setup", "fr_state_layout", "fr_rhs", "fr_set_state", "fr_get_state", "fr_rk_step", "fr_rk_run",
           "fr_rk_adaptive_run",
           "fr_sync", "fr_launch_count", "fr_profile_rhs", "fr_last_error", "fr_global_error", "fr_destroy",
           "fr_gemm", "fr_gemm_plan_create", "fr_gemm_plan_run", "fr_gemm_plan_destroy", "fr_probe_peaks", "fr_probe_dmma",
           "fr_profile_stage_kernels", "fr_check_finite", "fr_plan_describe", "fr_rhs_phase", "fr_rk_stage_phase",
           "fr_halo_buffers", "fr_halo_set_peers", "fr_gemm_static", "fr_gemm_plan_describe", "fr_probe_fp32_paths"]

_lib = None


def load():
    """dlopen libfrb200.so (built by paper_1409_0405_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libfrb200.so is not built: run `python -m paper_1409_0405_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    lib.fr_setup.argtypes = [C.POINTER(fr_config), C.POINTER(vp)]
    lib.fr_state_layout.argtypes = [vp, C.c_int32, _i64p, _i64p]
    lib.fr_rhs.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]
    lib.fr_set_state.argtypes = [vp, C.POINTER(_dp)]
    lib.fr_get_state.argtypes = [vp, C.POINTER(_dp)]
    lib.fr_rk_step.argtypes = [vp, C.c_double]
    lib.fr_rk_run.argtypes = [vp, C.c_double, C.c_int64]
    lib.fr_rk_adaptive_run.argtypes = [vp, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int64,
                                       C.POINTER(fr_adapt_stats), _dp, _dp, C.c_int64]
    lib.fr_sync.argtypes = [vp]
    lib.fr_launch_count.argtypes = [vp]
    lib.fr_launch_count.restype = C.c_int64
    lib.fr_profile_rhs.argtypes = [vp, C.c_int32, _dp]
    lib.fr_profile_kernels.argtypes = [vp, C.c_int32, C.POINTER(fr_kernel_stat), C.c_int32, _i32p]
    lib.fr_rk_step_host.argtypes = [vp, C.c_double, C.POINTER(vp)]
    lib.fr_last_error.argtypes = [vp]
    lib.fr_last_error.restype = C.c_char_p
    lib.fr_global_error.argtypes = []
    lib.fr_global_error.restype = C.c_char_p
    lib.fr_destroy.argtypes = [vp]
    lib.fr_destroy.restype = None
    lib.fr_gemm.argtypes = [C.c_int32, C.c_int32, C.c_int64, C.c_double, _dp, vp, C.c_int64, C.c_double, vp,
                            C.c_int64, C.c_int, vp]
    lib.fr_gemm_static.argtypes = lib.fr_gemm.argtypes
    lib.fr_gemm_plan_create.argtypes = [C.c_int32, C.c_int32, _dp, C.c_int, C.POINTER(vp)]
    lib.fr_gemm_plan_run.argtypes = [vp, C.c_int64, C.c_double, vp, C.c_int64, C.c_double, vp, C.c_int64, vp]
    lib.fr_gemm_plan_destroy.argtypes = [vp]
    lib.fr_gemm_plan_describe.argtypes = [vp, C.c_char_p, C.c_int64]
    lib.fr_gemm_plan_destroy.restype = None
    lib.fr_probe_peaks.argtypes = [_dp, _dp, _dp]
    lib.fr_probe_dmma.argtypes = [_dp]
    lib.fr_probe_fp32_paths.argtypes = [_dp, _dp, _dp, _dp]
    lib.fr_profile_stage_kernels.argtypes = [vp, C.c_int32, C.POINTER(fr_kernel_stat), C.c_int32, _i32p]
    lib.fr_check_finite.argtypes = [vp, _i64p]
    lib.fr_plan_describe.argtypes = [vp, C.c_char_p, C.c_int64]
    lib.fr_rhs_phase.argtypes = [vp, C.c_int32, C.POINTER(vp), C.POINTER(vp)]
    lib.fr_rk_stage_phase.argtypes = [vp, C.c_double, C.c_int32, C.c_int32]
    lib.fr_halo_buffers.argtypes = [vp, C.c_int32, C.POINTER(vp), C.POINTER(vp), _i64p]
    lib.fr_halo_set_peers.argtypes = [vp, C.c_int32, _i64p, _i64p]
    _lib = lib
    return lib


class FrError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("frb200 status %d: %s" % (status, msg))
        self.status = status


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a, t):
    return a.ctypes.data_as(t)


_ETYPE = {"tet": FR_TET, "pri": FR_PRI, "hex": FR_HEX}
_BCTYPE = {"wall": FR_BC_NOSLIP_ISOTHERMAL_WALL, "farfield": FR_BC_CHAR_RIEMANN_INV}


class Context:
    """fr_ctx wrapper.  `case` is a dict as produced by fr_inputs.cases (operators, metrics, pairs, BCs, cfg)."""

    def __init__(self, case, prec="f64", stepper="rk45", mode="fused", stream=0):
        lib = load()
        self._lib = lib
        self._keep = []
        cfgd = case["cfg"]
        ne = len(case["eles"])
        eles = (fr_eles_desc * ne)()
        for i, e in enumerate(case["eles"]):
            d = eles[i]
            d.etype, d.order, d.nupts, d.nfpts, d.neles = _ETYPE[e["etype"]], e["order"], e["nupts"], e["nfpts"], e["neles"]
            d.affine = 1 if e["affine"] else 0
            for k in ("M0", "M132", "M3", "M460", "M6"):
                a = _f64(e[k])
                self._keep.append(a)
                setattr(d, k, _ptr(a, _dp))
            sm, rj = e["smats"], e["rcpdjac"]
            if e["affine"]:
                sm, rj = sm[:, :, 0, :], rj[0, :]
            sm, rj = _f64(sm), _f64(rj)
            self._keep += [sm, rj]
            d.smats, d.rcpdjac = _ptr(sm, _dp), _ptr(rj, _dp)
        ifc = case["ifc"]
        fd = fr_iface_desc()
        fd.npairs = len(ifc["l_et"])
        for k, t, ct in (("l_et", np.int32, _i32p), ("l_fpt", np.int32, _i32p), ("l_ele", np.int64, _i64p),
                         ("r_et", np.int32, _i32p), ("r_fpt", np.int32, _i32p), ("r_ele", np.int64, _i64p),
                         ("nl", np.float64, _dp), ("magl", np.float64, _dp), ("magr", np.float64, _dp)):
            a = np.ascontiguousarray(ifc[k], dtype=t)
            self._keep.append(a)
            setattr(fd, k, _ptr(a, ct))
        nb = len(case["bcs"])
        bcs = (fr_bc_desc * max(nb, 1))()
        for i, b in enumerate(case["bcs"]):
            d = bcs[i]
            d.type, d.nfpts = _BCTYPE[b["type"]], len(b["et"])
            for k, t, ct in (("et", np.int32, _i32p), ("fpt", np.int32, _i32p), ("ele", np.int64, _i64p),
                             ("n", np.float64, _dp), ("mag", np.float64, _dp)):
                a = np.ascontiguousarray(b[k], dtype=t)
                self._keep.append(a)
                setattr(d, k, _ptr(a, ct))
            for j, v in enumerate(b["params"]):
                d.params[j] = float(v)
        cfg = fr_config()
        cfg.system = FR_NAVIER_STOKES if cfgd["system"] == "ns" else FR_EULER
        cfg.prec = FR_F64 if prec == "f64" else FR_F32
        cfg.stepper = {"rk4": FR_RK4, "rk45": FR_RK45_2R, "euler": FR_EULER1}[stepper]
        cfg.mode = FR_MODE_FUSED if mode == "fused" else FR_MODE_UNFUSED
        cfg.gamma, cfg.mu, cfg.prandtl = cfgd["gamma"], cfgd.get("mu", 0.0), cfgd.get("prandtl", 0.72)
        cfg.ldg_beta, cfg.ldg_tau = cfgd.get("ldg_beta", 0.5), cfgd.get("ldg_tau", 0.1)
        cfg.netypes, cfg.eles, cfg.ifaces = ne, eles, C.pointer(fd)
        cfg.nbcs, cfg.bcs = nb, bcs
        cfg.cuda_stream = C.c_void_p(stream)
        self.halo = case.get("halo")
        if self.halo is not None:
            hd = fr_halo_desc()
            hd.nghost = int(self.halo["nghost"])
            for k, t, ct in (("et", np.int32, _i32p), ("fpt", np.int32, _i32p), ("ele", np.int64, _i64p)):
                a = np.ascontiguousarray(self.halo[k], dtype=t)
                self._keep.append(a)
                setattr(hd, k, _ptr(a, ct))
            self._keep.append(hd)
            cfg.halo = C.pointer(hd)
        self.prec = prec
        self.dtype = np.float64 if prec == "f64" else np.float32
        self.netypes = ne
        self.shapes = [(e["nupts"], 5, e["neles"]) for e in case["eles"]]
        h = C.c_void_p()
        st = lib.fr_setup(C.byref(cfg), C.byref(h))
        self._keep = []          # fr_setup copied everything it needs
        if st != FR_OK:
            raise FrError(st, lib.fr_global_error().decode())
        self._h = h
        if self.halo is not None:
            st_ = np.ascontiguousarray([p_["start"] for p_ in self.halo["peers"]], dtype=np.int64)
            ct_ = np.ascontiguousarray([p_["count"] for p_ in self.halo["peers"]], dtype=np.int64)
            self._check(lib.fr_halo_set_peers(h, len(st_), _ptr(st_, _i64p), _ptr(ct_, _i64p)))
        self.ld = []
        self.nbytes = []
        for t in range(ne):
            ld, nbytes = C.c_int64(), C.c_int64()
            self._check(lib.fr_state_layout(h, t, C.byref(ld), C.byref(nbytes)))
            self.ld.append(ld.value)
            self.nbytes.append(nbytes.value)

    def _check(self, st):
        if st != FR_OK:
            raise FrError(st, self._lib.fr_last_error(self._h).decode())

    def rhs(self, u_ptrs, dudt_ptrs):
        """fr_rhs on DEVICE pointers (ints), one per element type, in the fr_state_layout layout."""
        n = self.netypes
        up = (C.c_void_p * n)(*[C.c_void_p(int(p)) for p in u_ptrs])
        dp = (C.c_void_p * n)(*[C.c_void_p(int(p)) for p in dudt_ptrs])
        self._check(self._lib.fr_rhs(self._h, up, dp))

    def set_state(self, us):
        arrs = [_f64(u) for u in us]
        for a, s in zip(arrs, self.shapes):
            if a.shape != s:
                raise ValueError("state shape %s, expected %s" % (a.shape, s))
        self._check(self._lib.fr_set_state(self._h, (_dp * self.netypes)(*[_ptr(a, _dp) for a in arrs])))

    def get_state(self):
        arrs = [np.empty(s, dtype=np.float64) for s in self.shapes]
        self._check(self._lib.fr_get_state(self._h, (_dp * self.netypes)(*[_ptr(a, _dp) for a in arrs])))
        return arrs

    def rk_step(self, dt):
        self._check(self._lib.fr_rk_step(self._h, float(dt)))

    def rk_run(self, dt, nsteps):
        self._check(self._lib.fr_rk_run(self._h, float(dt), int(nsteps)))

    def rk_adaptive_run(self, t0, t1, dt_init, atol, rtol, max_attempts=10000):
        """fr_rk_adaptive_run: returns (stats dict, history list of (dt tried, err, accepted))."""
        st = fr_adapt_stats()
        cap = int(max_attempts)
        dts, errs = (C.c_double * cap)(), (C.c_double * cap)()
        rc = self._lib.fr_rk_adaptive_run(self._h, float(t0), float(t1), float(dt_init), float(atol), float(rtol), cap,
                                          C.byref(st), dts, errs, cap)
        n = int(st.accepted + st.rejected)
        hist = [(dts[i], errs[i], bool(errs[i] <= 1.0)) for i in range(n)]
        self._check(rc)
        return dict(accepted=int(st.accepted), rejected=int(st.rejected), t=float(st.t), dt_next=float(st.dt_next)), hist

    def sync(self):
        self._check(self._lib.fr_sync(self._h))

    def launch_count(self):
        return int(self._lib.fr_launch_count(self._h))

    def profile_rhs(self, reps=5):
        ms = (C.c_double * 4)()
        self._check(self._lib.fr_profile_rhs(self._h, reps, ms))
        return dict(gemm_ms=ms[0], pointwise_ms=ms[1], iface_ms=ms[2], total_ms=ms[3])

    def profile_kernels(self, reps=5):
        cap = 128
        arr = (fr_kernel_stat * cap)()
        n = C.c_int32()
        self._check(self._lib.fr_profile_kernels(self._h, reps, arr, cap, C.byref(n)))
        return [dict(name=arr[i].name.decode(), ms=arr[i].ms, alg_bytes=arr[i].alg_bytes, flops=arr[i].flops,
                     category=arr[i].category) for i in range(min(n.value, cap))]

    def rhs_phase(self, phase, u_ptrs, dudt_ptrs=None):
        """fr_rhs_phase: phase 0, 1 or 2 of the partitioned right-hand side (the caller exchanges the halo buffers in between)."""
        n = self.netypes
        u = (C.c_void_p * n)(*[C.c_void_p(int(p)) for p in u_ptrs])
        d = (C.c_void_p * n)(*[C.c_void_p(int(p)) for p in dudt_ptrs]) if dudt_ptrs is not None else None
        self._check(self._lib.fr_rhs_phase(self._h, int(phase), u, d))

    def rk_stage_phase(self, dt, stage, phase):
        self._check(self._lib.fr_rk_stage_phase(self._h, float(dt), int(stage), int(phase)))

    def halo_buffers(self, which):
        """(send pointer, receive pointer, number of values) of the U_f (which = 0) or G_f (which = 1) exchange buffers."""
        s_, r_, n = C.c_void_p(), C.c_void_p(), C.c_int64()
        self._check(self._lib.fr_halo_buffers(self._h, int(which), C.byref(s_), C.byref(r_), C.byref(n)))
        return s_.value or 0, r_.value or 0, int(n.value)

    def profile_stage_kernels(self, reps=5, cap=64):
        """fr_profile_stage_kernels: the per-kernel breakdown of the right-hand side as an RK stage runs it."""
        arr = (fr_kernel_stat * cap)()
        n = C.c_int32(0)
        self._check(self._lib.fr_profile_stage_kernels(self._h, reps, arr, cap, C.byref(n)))
        return [dict(name=arr[i].name.decode(), ms=arr[i].ms, alg_bytes=arr[i].alg_bytes, flops=arr[i].flops,
                     category=arr[i].category) for i in range(min(n.value, cap))]

    def check_finite(self):
        n = C.c_int64(0)
        self._check(self._lib.fr_check_finite(self._h, C.byref(n)))
        return int(n.value)

    def plan_describe(self):
        buf = C.create_string_buffer(8192)
        self._check(self._lib.fr_plan_describe(self._h, buf, 8192))
        return buf.value.decode()

    def rk_step_host(self, dt, host_ptrs):
        """fr_rk_step_host on HOST pointers (ints) in the device layout / precision."""
        hp = (C.c_void_p * self.netypes)(*[C.c_void_p(int(p)) for p in host_ptrs])
        self._check(self._lib.fr_rk_step_host(self._h, float(dt), hp))

    def close(self):
        if getattr(self, "_h", None):
            self._lib.fr_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def gemm(A, B_ptr, ldb, C_ptr, ldc, N, c1=1.0, c2=0.0, prec="f64", stream=0):
    """fr_gemm: C <- c1*A*B + c2*C with A a host FP64 [M,K] array and B, C device pointers."""
    lib = load()
    A = _f64(A)
    M, K = A.shape
    st = lib.fr_gemm(M, K, N, c1, _ptr(A, _dp), C.c_void_p(int(B_ptr)), ldb, c2, C.c_void_p(int(C_ptr)), ldc,
                     FR_F64 if prec == "f64" else FR_F32, C.c_void_p(stream))
    if st != FR_OK:
        raise FrError(st, lib.fr_global_error().decode())


def gemm_static(A, B_ptr, ldb, C_ptr, ldc, N, c1=1.0, c2=0.0, prec="f64", stream=0):
    """fr_gemm_static: fr_gemm without device allocations (packed operator in a static device array of GEMM_STATIC_MAX_BYTES)."""
    lib = load()
    A = _f64(A)
    M, K = A.shape
    st = lib.fr_gemm_static(M, K, N, c1, _ptr(A, _dp), C.c_void_p(int(B_ptr)), ldb, c2, C.c_void_p(int(C_ptr)), ldc,
                            FR_F64 if prec == "f64" else FR_F32, C.c_void_p(stream))
    if st != FR_OK:
        raise FrError(st, lib.fr_global_error().decode())


class GemmPlan:
    def __init__(self, A, prec="f64"):
        lib = load()
        A = _f64(A)
        self._lib, self.M, self.K = lib, A.shape[0], A.shape[1]
        h = C.c_void_p()
        st = lib.fr_gemm_plan_create(self.M, self.K, _ptr(A, _dp), FR_F64 if prec == "f64" else FR_F32, C.byref(h))
        if st != FR_OK:
            raise FrError(st, lib.fr_global_error().decode())
        self._h = h

    def describe(self):
        """fr_gemm_plan_describe: one line per launch (packing, streamed or resident operator, geometry)."""
        buf = C.create_string_buffer(8192)
        st = self._lib.fr_gemm_plan_describe(self._h, buf, len(buf))
        if st != FR_OK:
            raise FrError(st, self._lib.fr_global_error().decode())
        return buf.value.decode()

    def run(self, B_ptr, ldb, C_ptr, ldc, N, c1=1.0, c2=0.0, stream=0):
        st = self._lib.fr_gemm_plan_run(self._h, N, c1, C.c_void_p(int(B_ptr)), ldb, c2, C.c_void_p(int(C_ptr)), ldc,
                                        C.c_void_p(stream))
        if st != FR_OK:
            raise FrError(st, self._lib.fr_global_error().decode())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.fr_gemm_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def probe_dmma():
    """fr_probe_dmma: TFLOP/s of the FP64 tensor pipe (mma.sync.m8n8k4.f64 chains)."""
    lib = load()
    a = C.c_double()
    st = lib.fr_probe_dmma(C.byref(a))
    if st != FR_OK:
        raise FrError(st, "fr_probe_dmma failed")
    return a.value


def probe_fp32_paths():
    """fr_probe_fp32_paths: TFLOP/s of FFMA2 chains, FFMA / FFMA2 chains with integer work beside them, and mma.sync TF32."""
    lib = load()
    v = [C.c_double() for _ in range(4)]
    st = lib.fr_probe_fp32_paths(*[C.byref(x) for x in v])
    if st != FR_OK:
        raise FrError(st, "fr_probe_fp32_paths failed")
    return dict(zip(("ffma2_tflops", "ffma_mixed_tflops", "ffma2_mixed_tflops", "tf32_mma_tflops"), (x.value for x in v)))


def probe_peaks():
    lib = load()
    a, b, c = C.c_double(), C.c_double(), C.c_double()
    st = lib.fr_probe_peaks(C.byref(a), C.byref(b), C.byref(c))
    if st != FR_OK:
        raise FrError(st, "fr_probe_peaks failed")
    return dict(fp64_tflops=a.value, fp32_tflops=b.value, copy_gbs=c.value)
