"""Thin ctypes binding of libgenga_kick.so (include/genga_kick.h, include/genga_step.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the library's CUDA
kernels.  There is no CPU fallback: if the library is missing or no sm_100 device is present the
calls raise."""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libgenga_kick.so")

OK, E_NULL, E_ALIGN, E_SIZE, E_LEVEL, E_CUDA, E_NOMEM = 0, -1, -2, -3, -4, -5, -6
STATUS_COINCIDENT = 1
STATUS_CAND_OVERFLOW = 2
STATUS_FX_RANGE = 4
ORDER_AUTO, ORDER_CALLER, ORDER_SORTED = 0, 1, 2

EXPORTS = (
    "genga_kick_make_plan", "genga_kick_make_plan_tp2", "genga_kick_make_plan_sym", "genga_kick_make_plan_tprows",
    "genga_kick_plan_sym_row_begin", "genga_kick_plan_sym_row_of", "genga_kick_plan_sym_table", "genga_kick_plan_cta_range", "genga_kick_plan_iblock_ctas", "genga_kick_init",
    "genga_kick_set_stream", "genga_kick", "genga_kick_set_order_reuse", "genga_kick_list", "genga_kick_host", "genga_kick_get_plan", "genga_kick_status",
    "genga_kick_launch_count", "genga_kick_free", "genga_kick_strerror", "genga_kick_last_cuda_error",
    "genga_kick_enable_timing", "genga_kick_last_pair_loop_ms",
)
# include/genga_step.h: the O(N) neighbours of the kick and the composed step
STEP_EXPORTS = ("genga_rcrit", "genga_hc", "genga_fg", "genga_drift", "genga_step", "genga_rcrit_list", "genga_fg_list")
# include/genga_group.h: close-encounter groups
GROUP_EXPORTS = ("genga_group",)
STATUS_BAD_PAIR = 16
# include/genga_bs.h: Bulirsch-Stoer integration of the groups
BS_EXPORTS = ("genga_bs", "genga_hybrid_step", "genga_bs_set_stats", "genga_bs_totals")
STATUS_GROUP_TOO_LARGE, STATUS_BS_NOT_CONVERGED = 32, 64
STATUS_UNBOUND = 8
# include/genga_senc.h: close-encounter detection and the multi-level step (SEnc)
SENC_EXPORTS = ("genga_detect", "genga_multilevel_step", "genga_steps")
STATUS_RCRIT_JUMP = 256
REUSE_OFF, REUSE_ORDER, REUSE_LIST = 0, 1, 2
STATUS_LIST_CLIPPED = 128
# include/genga_kick_static.h: the list kick without a context and without any allocation
STATIC_EXPORTS = ("genga_kick_list_static",)
STATIC_MAX_BODIES = 65536
E_STATIC_MAX = -7


class GengaKickConfig(C.Structure):
    _fields_ = [("n_massive", C.c_int32), ("n_test", C.c_int32), ("max_level", C.c_int32), ("device", C.c_int32),
                ("pair_capacity", C.c_int64), ("G", C.c_double), ("enc_factor", C.c_double),
                ("order_mode", C.c_int32), ("tp_mode", C.c_int32)]


class GengaSencConfig(C.Structure):
    _fields_ = [("slevels", C.c_int32), ("substeps", C.c_int32), ("detect", C.c_int32), ("reserved", C.c_int32),
                ("n1", C.c_double), ("n2", C.c_double), ("tol", C.c_double)]


class GengaKickPlan(C.Structure):
    _fields_ = [("threads", C.c_int32), ("i_per_thread", C.c_int32), ("i_block", C.c_int32), ("j_tile", C.c_int32),
                ("m_pad", C.c_int32), ("n_i_blocks", C.c_int32), ("n_j_tiles", C.c_int32), ("n_tiles", C.c_int64),
                ("n_ctas", C.c_int32), ("max_segs", C.c_int32), ("n_rec", C.c_int64), ("partial_doubles", C.c_int64),
                ("symmetric", C.c_int32), ("tiles_per_iblock", C.c_int32), ("react_doubles", C.c_int64)]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


class GengaKickError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"genga_kick error {code}: {text}")
        self.code = code


_lib = None


def lib():
    """The loaded C-ABI library.  Raises if it has not been built (python -m paper_2201_10058_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2201_10058_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, d = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        L.genga_kick_make_plan.argtypes = [i32, i32, i32, i32, C.POINTER(GengaKickPlan)]
        L.genga_kick_make_plan_tp2.argtypes = [i32, i32, i32, C.POINTER(GengaKickPlan)]
        L.genga_kick_make_plan_sym.argtypes = [i32, i32, i32, C.POINTER(GengaKickPlan)]
        L.genga_kick_make_plan_tprows.argtypes = [i32, i32, i32, C.POINTER(GengaKickPlan)]
        L.genga_kick_plan_sym_table.argtypes = [C.POINTER(GengaKickPlan), vp]
        L.genga_kick_plan_sym_row_begin.argtypes = [C.POINTER(GengaKickPlan), i32]
        L.genga_kick_plan_sym_row_begin.restype = i64
        L.genga_kick_plan_sym_row_of.argtypes = [C.POINTER(GengaKickPlan), i64]
        L.genga_kick_plan_sym_row_of.restype = i32
        L.genga_kick_plan_cta_range.argtypes = [C.POINTER(GengaKickPlan), i32, C.POINTER(i64), C.POINTER(i64)]
        L.genga_kick_plan_iblock_ctas.argtypes = [C.POINTER(GengaKickPlan), i32, C.POINTER(i32), C.POINTER(i32)]
        L.genga_kick_init.argtypes = [C.POINTER(GengaKickConfig), C.POINTER(vp)]
        L.genga_kick_set_stream.argtypes = [vp, vp]
        L.genga_kick_set_order_reuse.argtypes = [vp, i32]
        L.genga_kick.argtypes = [vp, vp, vp, vp, vp, i32, d, vp, vp, vp]
        L.genga_kick_list.argtypes = [vp, vp, vp, vp, vp, i32, d, vp, vp, i64, vp, vp, vp]
        L.genga_kick_host.argtypes = [vp, vp, vp, vp, vp, i32, d, vp, vp, vp]
        L.genga_kick_get_plan.argtypes = [vp, i32, C.POINTER(GengaKickPlan)]
        L.genga_kick_status.argtypes = [vp, C.POINTER(i32)]
        L.genga_kick_launch_count.argtypes = [vp]
        L.genga_kick_enable_timing.argtypes = [vp, i32]
        L.genga_kick_last_pair_loop_ms.argtypes = [vp, i32, C.POINTER(C.c_float)]
        L.genga_kick_launch_count.restype = i64
        L.genga_kick_free.argtypes = [vp]
        L.genga_kick_strerror.argtypes = [C.c_int]
        L.genga_kick_strerror.restype = C.c_char_p
        L.genga_kick_last_cuda_error.argtypes = [vp]
        L.genga_kick_last_cuda_error.restype = C.c_char_p
        L.genga_rcrit.argtypes = [vp, vp, vp, vp, d, d, d, i32, d, d, vp]
        L.genga_hc.argtypes = [vp, vp, vp, vp, d, d]
        L.genga_fg.argtypes = [vp, vp, vp, d, d]
        L.genga_drift.argtypes = [vp, vp, vp, vp, d, d]
        L.genga_rcrit_list.argtypes = [vp, vp, vp, vp, d, d, d, i32, d, d, vp, vp, i64, vp]
        L.genga_fg_list.argtypes = [vp, vp, vp, d, d, vp, vp, i64]
        L.genga_step.argtypes = [vp, vp, vp, vp, d, d, d, d, vp, vp, vp, vp]
        L.genga_group.argtypes = [vp, vp, vp, i64, vp, vp, vp, vp]
        L.genga_hybrid_step.argtypes = [vp, vp, vp, vp, d, d, d, d, d, vp, vp, vp, vp, vp, vp, vp]
        L.genga_bs.argtypes = [vp, vp, vp, vp, vp, i32, d, d, d, vp, vp, vp, vp, vp]
        L.genga_bs_set_stats.argtypes = [vp, vp, i64]
        L.genga_bs_totals.argtypes = [vp, C.POINTER(i64 * 4), i32]
        L.genga_detect.argtypes = [vp, vp, vp, vp, vp, vp, d, d, vp, vp, i64, vp, vp]
        L.genga_multilevel_step.argtypes = [vp, vp, vp, vp, d, d, C.POINTER(GengaSencConfig), vp, vp, vp, vp]
        L.genga_steps.argtypes = [vp, vp, vp, vp, d, d, i32, C.POINTER(GengaSencConfig), vp, vp, vp, vp]
        L.genga_kick_list_static.argtypes = [vp, vp, vp, vp, i64, i64, i32, i32, d, d, d, vp, vp, i64, vp, vp, i64, vp, vp, vp]
        for name in EXPORTS + STEP_EXPORTS + GROUP_EXPORTS + BS_EXPORTS + SENC_EXPORTS + STATIC_EXPORTS:
            if name not in ("genga_kick_launch_count", "genga_kick_strerror", "genga_kick_last_cuda_error",
                            "genga_kick_plan_sym_row_begin", "genga_kick_plan_sym_row_of"):
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def strerror(code: int) -> str:
    return lib().genga_kick_strerror(int(code)).decode()


def kick_list_static(pos, vel, mass, rcrit, n_massive, n_test, changeover_level, dt, in_pairs, in_n_pairs, in_pair_rows,
                     out_acc, out_pairs, out_npairs, status, G=1.0, enc_factor=1.0, tp_mode=1, cuda_stream=0):
    """include/genga_kick_static.h: genga_kick_list with the scratch in a static device array of the library -- no
    context, no allocation, N <= STATIC_MAX_BODIES; calls that overlap on the GPU race on that array.  `status`: one
    int32 on the device (out).  out_pairs: [capacity, 2] int32 or None."""
    n = int(n_massive) + int(n_test)
    cap = 0 if out_pairs is None else int(out_pairs.numel()) // 2
    rows = max(int(changeover_level), 0) + 1
    rc = lib().genga_kick_list_static(
        _ptr(pos, "f8", 3 * n, "pos"), _ptr(vel, "f8", 3 * n, "vel"), _ptr(mass, "f8", n, "mass"),
        _ptr(rcrit, "f8", rows * n, "rcrit"), int(n_massive), int(n_test), int(changeover_level), int(tp_mode), float(G),
        float(enc_factor), float(dt), _ptr(in_pairs, "i4", 2 * int(in_pair_rows), "in_pairs"),
        _ptr(in_n_pairs, "i4", 1, "in_n_pairs"), int(in_pair_rows), _ptr(out_acc, "f8", 3 * n, "out_acc"),
        _ptr(out_pairs, "i4", 2 * cap, "out_pairs"), cap, _ptr(out_npairs, "i4", n + 1, "out_npairs"),
        _ptr(status, "i4", 1, "status"), C.c_void_p(int(cuda_stream)))
    if rc != OK:
        raise GengaKickError(rc, strerror(rc))


def make_plan(n_massive: int, n_test: int, level: int, num_sms: int) -> GengaKickPlan:
    plan = GengaKickPlan()
    rc = lib().genga_kick_make_plan(n_massive, n_test, level, num_sms, C.byref(plan))
    if rc != OK:
        raise GengaKickError(rc, strerror(rc))
    return plan


def make_plan_tp2(n_massive: int, n_test: int, num_sms: int) -> GengaKickPlan:
    plan = GengaKickPlan()
    rc = lib().genga_kick_make_plan_tp2(n_massive, n_test, num_sms, C.byref(plan))
    if rc != OK:
        raise GengaKickError(rc, strerror(rc))
    return plan


def make_plan_sym(n_massive: int, n_test: int, num_sms: int) -> GengaKickPlan:
    plan = GengaKickPlan()
    rc = lib().genga_kick_make_plan_sym(n_massive, n_test, num_sms, C.byref(plan))
    if rc != OK:
        raise GengaKickError(rc, strerror(rc))
    return plan


def make_plan_tprows(n_massive: int, n_test: int, num_sms: int) -> GengaKickPlan:
    plan = GengaKickPlan()
    rc = lib().genga_kick_make_plan_tprows(n_massive, n_test, num_sms, C.byref(plan))
    if rc != OK:
        raise GengaKickError(rc, strerror(rc))
    return plan


def plan_sym_row_begin(plan: GengaKickPlan, row: int) -> int:
    return int(lib().genga_kick_plan_sym_row_begin(C.byref(plan), int(row)))


def plan_sym_row_of(plan: GengaKickPlan, t: int) -> int:
    return int(lib().genga_kick_plan_sym_row_of(C.byref(plan), int(t)))


def plan_cta_range(plan: GengaKickPlan, cta: int):
    t0, t1 = C.c_int64(), C.c_int64()
    rc = lib().genga_kick_plan_cta_range(C.byref(plan), cta, C.byref(t0), C.byref(t1))
    if rc != OK:
        raise GengaKickError(rc, strerror(rc))
    return t0.value, t1.value


def plan_iblock_ctas(plan: GengaKickPlan, ib: int):
    a, b = C.c_int32(), C.c_int32()
    rc = lib().genga_kick_plan_iblock_ctas(C.byref(plan), ib, C.byref(a), C.byref(b))
    if rc != OK:
        raise GengaKickError(rc, strerror(rc))
    return a.value, b.value


def _ptr(t, dtype=None, numel=0, name="array", host=False):
    """Pointer of a tensor for the C ABI, after the checks the library cannot make on a bare pointer: the side it
    lives on (device for every call but kick_host), dtype ("f8" / "i4"), C-contiguity and at least `numel` elements.
    None stays NULL (the library decides whether that argument is optional)."""
    if t is None:
        return None
    if host == bool(getattr(t, "is_cuda", False)):
        raise ValueError(f"{name}: expected a {'CPU' if host else 'CUDA device'} tensor")
    if dtype is not None:
        import torch
        want = torch.float64 if dtype == "f8" else torch.int32
        if t.dtype != want:
            raise TypeError(f"{name}: expected dtype {want}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError(f"{name}: expected a C-contiguous tensor")
    if t.numel() < numel:
        raise ValueError(f"{name}: expected at least {numel} elements, got {t.numel()}")
    return C.c_void_p(t.data_ptr())


class GengaKick:
    """A genga_kick context.  Arrays are torch tensors (device tensors for kick(), CPU tensors for
    kick_host()), float64 / int32, C-contiguous, laid out as include/genga_kick.h states."""

    def __init__(self, n_massive, n_test=0, max_level=0, pair_capacity=1 << 20, G=1.0, enc_factor=1.0, device=0,
                 order_mode=0, tp_mode=1):
        self.cfg = GengaKickConfig(int(n_massive), int(n_test), int(max_level), int(device), int(pair_capacity),
                                   float(G), float(enc_factor), int(order_mode), int(tp_mode))
        self.n = int(n_massive) + int(n_test)
        self._ctx = C.c_void_p()
        rc = lib().genga_kick_init(C.byref(self.cfg), C.byref(self._ctx))
        if rc != OK:
            raise GengaKickError(rc, strerror(rc))

    def _check(self, rc):
        if rc != OK:
            text = strerror(rc)
            if rc == E_CUDA:
                text += ": " + lib().genga_kick_last_cuda_error(self._ctx).decode()
            raise GengaKickError(rc, text)

    def set_stream(self, cuda_stream: int):
        self._check(lib().genga_kick_set_stream(self._ctx, C.c_void_p(int(cuda_stream))))

    def _kick_args(self, pos, vel, mass, rcrit, level, out_acc, out_pairs, out_npairs, host=False):
        n, cap = self.n, int(self.cfg.pair_capacity)
        rows = max(int(level), 0) + 1
        return (_ptr(pos, "f8", 3 * n, "pos", host), _ptr(vel, "f8", 3 * n, "vel", host), _ptr(mass, "f8", n, "mass", host),
                _ptr(rcrit, "f8", rows * n, "rcrit", host), _ptr(out_acc, "f8", 3 * n, "out_acc", host),
                _ptr(out_pairs, "i4", 2 * cap, "out_pairs", host), _ptr(out_npairs, "i4", n + 1, "out_npairs", host))

    def set_order_reuse(self, on):
        """0 / False: off; 1 / True: keep the internal order (REUSE_ORDER); 2: also the level-0 list of near pairs (REUSE_LIST)"""
        self._check(lib().genga_kick_set_order_reuse(self._ctx, int(on)))

    def kick(self, pos, vel, mass, rcrit, changeover_level, dt, out_acc, out_pairs, out_npairs):
        p, v, m, rc, a, op, on = self._kick_args(pos, vel, mass, rcrit, changeover_level, out_acc, out_pairs, out_npairs)
        self._check(lib().genga_kick(self._ctx, p, v, m, rc, int(changeover_level), float(dt), a, op, on))

    def kick_list(self, pos, vel, mass, rcrit, changeover_level, dt, in_pairs, in_n_pairs, in_pair_rows, out_acc,
                  out_pairs, out_npairs):
        p, v, m, rc, a, op, on = self._kick_args(pos, vel, mass, rcrit, changeover_level, out_acc, out_pairs, out_npairs)
        self._check(lib().genga_kick_list(self._ctx, p, v, m, rc, int(changeover_level), float(dt),
                                          _ptr(in_pairs, "i4", 2 * int(in_pair_rows), "in_pairs"),
                                          _ptr(in_n_pairs, "i4", 1, "in_n_pairs"), int(in_pair_rows), a, op, on))

    def kick_host(self, pos, vel, mass, rcrit, changeover_level, dt, out_acc, out_pairs, out_npairs):
        p, v, m, rc, a, op, on = self._kick_args(pos, vel, mass, rcrit, changeover_level, out_acc, out_pairs, out_npairs,
                                                 host=True)
        self._check(lib().genga_kick_host(self._ctx, p, v, m, rc, int(changeover_level), float(dt), a, op, on))

    # include/genga_step.h
    def _f(self, t, numel, name):
        return _ptr(t, "f8", numel, name)

    def _i(self, t, numel, name):
        return _ptr(t, "i4", numel, name)

    def rcrit(self, pos, vel, mass, m_star, dt, out_rcrit, substeps=2.0, nrows=1, n1=3.0, n2=0.4):
        n = self.n
        self._check(lib().genga_rcrit(self._ctx, self._f(pos, 3 * n, "pos"), self._f(vel, 3 * n, "vel"),
                                      self._f(mass, n, "mass"), float(m_star), float(dt), float(substeps), int(nrows),
                                      float(n1), float(n2), self._f(out_rcrit, max(int(nrows), 0) * n, "out_rcrit")))

    def hc(self, pos, vel, mass, m_star, dt):
        n = self.n
        self._check(lib().genga_hc(self._ctx, self._f(pos, 3 * n, "pos"), self._f(vel, 3 * n, "vel"),
                                   self._f(mass, n, "mass"), float(m_star), float(dt)))

    def fg(self, pos, vel, m_star, dt):
        n = self.n
        self._check(lib().genga_fg(self._ctx, self._f(pos, 3 * n, "pos"), self._f(vel, 3 * n, "vel"), float(m_star),
                                   float(dt)))

    def rcrit_list(self, pos, vel, mass, m_star, dt, list_, n_list, list_rows, out_rcrit, substeps=2.0, nrows=1, n1=3.0,
                   n2=0.4):
        n = self.n
        self._check(lib().genga_rcrit_list(self._ctx, self._f(pos, 3 * n, "pos"), self._f(vel, 3 * n, "vel"),
                                           self._f(mass, n, "mass"), float(m_star), float(dt), float(substeps), int(nrows),
                                           float(n1), float(n2), self._i(list_, int(list_rows), "list"),
                                           self._i(n_list, 1, "n_list"), int(list_rows),
                                           self._f(out_rcrit, max(int(nrows), 0) * n, "out_rcrit")))

    def fg_list(self, pos, vel, m_star, dt, list_, n_list, list_rows):
        n = self.n
        self._check(lib().genga_fg_list(self._ctx, self._f(pos, 3 * n, "pos"), self._f(vel, 3 * n, "vel"), float(m_star),
                                        float(dt), self._i(list_, int(list_rows), "list"), self._i(n_list, 1, "n_list"),
                                        int(list_rows)))

    def drift(self, pos, vel, mass, m_star, dt):
        n = self.n
        self._check(lib().genga_drift(self._ctx, self._f(pos, 3 * n, "pos"), self._f(vel, 3 * n, "vel"),
                                      self._f(mass, n, "mass"), float(m_star), float(dt)))

    def _step_args(self, pos, vel, mass, out_acc, out_pairs, out_npairs):
        n, cap = self.n, int(self.cfg.pair_capacity)
        return (self._f(pos, 3 * n, "pos"), self._f(vel, 3 * n, "vel"), self._f(mass, n, "mass"),
                self._f(out_acc, 3 * n, "out_acc"), self._i(out_pairs, 2 * cap, "out_pairs"),
                self._i(out_npairs, n + 1, "out_npairs"))

    def step(self, pos, vel, mass, m_star, dt, rcrit_row, out_acc, out_pairs, out_npairs, n1=3.0, n2=0.4):
        p, v, m, a, op, on = self._step_args(pos, vel, mass, out_acc, out_pairs, out_npairs)
        self._check(lib().genga_step(self._ctx, p, v, m, float(m_star), float(dt), float(n1), float(n2),
                                     self._f(rcrit_row, self.n, "rcrit_row"), a, op, on))

    # include/genga_group.h
    def _group_args(self, group_of, members, offsets, summary):
        n = self.n
        return (self._i(group_of, n, "group_of"), self._i(members, n, "members"), self._i(offsets, n + 1, "offsets"),
                self._i(summary, 4, "summary"))

    def group(self, pairs, n_pairs, pair_rows, group_of, members, offsets, summary):
        """n_pairs: a device int32 tensor VIEW whose first element is the pair count (e.g. out_npairs[N:])."""
        self._check(lib().genga_group(self._ctx, self._i(pairs, 2 * int(pair_rows), "pairs"), self._i(n_pairs, 1, "n_pairs"),
                                      int(pair_rows), *self._group_args(group_of, members, offsets, summary)))

    # include/genga_bs.h
    def bs(self, pos_in, vel_in, mass, rcrit, nlevels, m_star, dt, tol, members, offsets, summary, pos, vel):
        n = self.n
        self._check(lib().genga_bs(self._ctx, self._f(pos_in, 3 * n, "pos_in"), self._f(vel_in, 3 * n, "vel_in"),
                                   self._f(mass, n, "mass"), self._f(rcrit, max(int(nlevels), 0) * n, "rcrit"), int(nlevels),
                                   float(m_star), float(dt), float(tol), self._i(members, n, "members"),
                                   self._i(offsets, n + 1, "offsets"), self._i(summary, 4, "summary"),
                                   self._f(pos, 3 * n, "pos"), self._f(vel, 3 * n, "vel")))

    def bs_set_stats(self, group_stats, rows):
        self._check(lib().genga_bs_set_stats(self._ctx, self._i(group_stats, 4 * int(rows), "group_stats"), int(rows)))

    def bs_totals(self, reset=False):
        """(accepted macro steps, rejected attempts, force evaluations, groups integrated) since init / the last reset."""
        t = (C.c_int64 * 4)()
        self._check(lib().genga_bs_totals(self._ctx, C.byref(t), 1 if reset else 0))
        return tuple(int(x) for x in t)

    def hybrid_step(self, pos, vel, mass, m_star, dt, tol, out_acc, out_pairs, out_npairs, group_of, members, offsets,
                    summary, n1=3.0, n2=0.4):
        p, v, m, a, op, on = self._step_args(pos, vel, mass, out_acc, out_pairs, out_npairs)
        self._check(lib().genga_hybrid_step(self._ctx, p, v, m, float(m_star), float(dt), float(n1), float(n2), float(tol),
                                            a, op, on, *self._group_args(group_of, members, offsets, summary)))

    # include/genga_senc.h
    def detect(self, pos0, vel0, pos1, vel1, rcrit_row, h, in_pairs, in_n_pairs, in_pair_rows, out_pairs, out_npairs,
               enc_factor=1.0):
        n, cap = self.n, int(self.cfg.pair_capacity)
        self._check(lib().genga_detect(self._ctx, self._f(pos0, 3 * n, "pos0"), self._f(vel0, 3 * n, "vel0"),
                                       self._f(pos1, 3 * n, "pos1"), self._f(vel1, 3 * n, "vel1"),
                                       self._f(rcrit_row, n, "rcrit_row"), float(enc_factor), float(h),
                                       self._i(in_pairs, 2 * int(in_pair_rows), "in_pairs"),
                                       self._i(in_n_pairs, 1, "in_n_pairs"), int(in_pair_rows),
                                       self._i(out_pairs, 2 * cap, "out_pairs"), self._i(out_npairs, n + 1, "out_npairs")))

    def multilevel_step(self, pos, vel, mass, m_star, dt, slevels, substeps, tol, out_acc, out_pairs, out_npairs,
                        out_stats, detect=True, n1=3.0, n2=0.4):
        cfg = GengaSencConfig(int(slevels), int(substeps), int(bool(detect)), 0, float(n1), float(n2), float(tol))
        p, v, m, a, op, on = self._step_args(pos, vel, mass, out_acc, out_pairs, out_npairs)
        self._check(lib().genga_multilevel_step(self._ctx, p, v, m, float(m_star), float(dt), C.byref(cfg), a, op, on,
                                                self._i(out_stats, 4 * max(int(slevels), 0), "out_stats")))

    def steps(self, pos, vel, mass, m_star, dt, n_steps, slevels, substeps, tol, out_acc, out_pairs, out_npairs, out_stats,
              detect=True, n1=3.0, n2=0.4):
        """n_steps consecutive steps with merged kicks (include/genga_senc.h); slevels = 0: no encounter branch."""
        cfg = GengaSencConfig(int(slevels), int(substeps), int(bool(detect)), 0, float(n1), float(n2), float(tol))
        p, v, m, a, op, on = self._step_args(pos, vel, mass, out_acc, out_pairs, out_npairs)
        self._check(lib().genga_steps(self._ctx, p, v, m, float(m_star), float(dt), int(n_steps), C.byref(cfg), a, op, on,
                                      self._i(out_stats, 4 * max(int(slevels), 0), "out_stats")))

    def plan(self, changeover_level=0) -> GengaKickPlan:
        plan = GengaKickPlan()
        self._check(lib().genga_kick_get_plan(self._ctx, int(changeover_level), C.byref(plan)))
        return plan

    def status(self) -> int:
        s = C.c_int32()
        self._check(lib().genga_kick_status(self._ctx, C.byref(s)))
        return s.value

    def launch_count(self) -> int:
        return int(lib().genga_kick_launch_count(self._ctx))

    def enable_timing(self, on=True):
        self._check(lib().genga_kick_enable_timing(self._ctx, 1 if on else 0))

    def last_pair_loop_ms(self, changeover_level=0) -> float:
        ms = C.c_float()
        self._check(lib().genga_kick_last_pair_loop_ms(self._ctx, int(changeover_level), C.byref(ms)))
        return float(ms.value)

    def free(self):
        if self._ctx:
            lib().genga_kick_free(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass
