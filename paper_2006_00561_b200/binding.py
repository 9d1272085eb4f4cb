"""ctypes binding of libpa_b200.so (include/pa_b200.h): argument marshalling only.

PyTorch is used for device memory (the workspace tensor) and the stream; every step of the path runs in
the library's CUDA kernels.  There is no CPU fallback: a missing library or a missing GPU raises.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libpa_b200.so")

PA_OK, PA_EINVAL, PA_ENOMEM, PA_ECAPACITY, PA_EEXTINCT, PA_ECUDA = 0, -1, -2, -3, -4, -5
PA_KEEP_TAU, PA_KEEP_COUNTS, PA_PROFILE, PA_PROFILE_SPAN, PA_RESAMPLE_NEAREST, PA_RESAMPLE_SYSTEMATIC = 1, 2, 4, 8, 16, 32
PA_POLICY_BALANCED, PA_POLICY_MAIN, PA_POLICY_NAIVE, PA_POLICY_NONE = 0, 1, 2, 3
KERNELS = ["levels_w", "q_reduce", "levels_tau", "poisson_scan", "balance", "copy", "sweep", "observe", "resample_span"]

EXPORTS = ["pa_workspace_bytes", "pa_init", "pa_step", "pa_run", "pa_adaptive_beta", "pa_population", "pa_beta", "pa_totals", "pa_energies", "pa_log_Z",
           "pa_observables", "pa_spins", "pa_tau", "pa_counts", "pa_parents", "pa_partitions", "pa_thresholds",
           "pa_set_spins", "pa_debug_set_thresholds", "pa_set_bonds", "pa_overlap_hist", "pa_overlap_hist_static", "pa_static_last_error", "pa_dist_init", "pa_dist_workspace_bytes", "pa_dist_begin",
           "pa_dist_resample", "pa_dist_exchange_plan", "pa_dist_plan_check", "pa_dist_capacity", "pa_dist_pack", "pa_dist_buffers", "pa_dist_finish", "pa_dist_new_count",
           "pa_dist_abort", "pa_profile_read", "pa_launch_count", "pa_last_error", "pa_destroy"]


class PaConfig(C.Structure):
    _fields_ = [("L", C.c_int32), ("P", C.c_int32), ("R0", C.c_int64), ("capacity", C.c_int64), ("seed", C.c_uint64),
                ("beta0", C.c_double), ("workspace", C.c_void_p), ("workspace_bytes", C.c_uint64),
                ("stream", C.c_void_p), ("flags", C.c_uint32), ("policy", C.c_uint32), ("block", C.c_uint32),
                ("maxexc", C.c_uint32)]


class PaObs(C.Structure):
    _fields_ = [("R", C.c_int64), ("sum_E", C.c_int64), ("sum_E2", C.c_uint64 * 2), ("sum_absM", C.c_uint64 * 2),
                ("sum_M2", C.c_uint64 * 2), ("sum_M4", C.c_uint64 * 2), ("mean_E", C.c_double), ("mean_E2", C.c_double),
                ("mean_absM", C.c_double), ("mean_M2", C.c_double), ("mean_M4", C.c_double)]


class PaDistPartial(C.Structure):
    _fields_ = [("sumw", C.c_double), ("R", C.c_int64)]


class PaError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("pa_b200 error %d: %s" % (code, msg))
        self.code = code


_lib = None


def load_library():
    """dlopen libpa_b200.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libpa_b200.so is not built (run `python -m paper_2006_00561_b200.build`); "
                          "there is no CPU fallback")
    lib = C.CDLL(LIB_PATH)
    vp, i64p, i32p, u32p, f64p = C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int32), C.POINTER(C.c_uint32), \
        C.POINTER(C.c_double)
    proto = {
        "pa_workspace_bytes": (C.c_uint64, [C.POINTER(PaConfig)]),
        "pa_init": (C.c_int, [C.POINTER(PaConfig), C.POINTER(vp)]),
        "pa_step": (C.c_int, [vp, C.c_double, C.c_int32]),
        "pa_run": (C.c_int, [vp, f64p, C.c_int32, C.c_int32, i32p]),
        "pa_adaptive_beta": (C.c_int, [vp, C.c_double, C.c_double, f64p]),
        "pa_population": (C.c_int, [vp, i64p]),
        "pa_beta": (C.c_int, [vp, f64p, i64p]),
        "pa_totals": (C.c_int, [vp, i64p]),
        "pa_energies": (C.c_int, [vp, vp, vp, C.c_int64, C.c_int]),
        "pa_log_Z": (C.c_int, [vp, f64p, f64p, f64p]),
        "pa_observables": (C.c_int, [vp, C.POINTER(PaObs)]),
        "pa_spins": (C.c_int, [vp, vp, C.c_int64, C.c_int64, C.c_int]),
        "pa_tau": (C.c_int, [vp, vp, C.c_int64, C.c_int]),
        "pa_counts": (C.c_int, [vp, vp, vp, C.c_int64, C.c_int]),
        "pa_parents": (C.c_int, [vp, i64p]),
        "pa_partitions": (C.c_int, [vp, vp, vp, i64p]),
        "pa_thresholds": (C.c_int, [vp, u32p, u32p]),
        "pa_set_spins": (C.c_int, [vp, vp, C.c_int64, C.c_int]),
        "pa_debug_set_thresholds": (C.c_int, [vp, C.c_int, C.c_uint32, C.c_uint32]),
        "pa_set_bonds": (C.c_int, [vp, vp, vp]),
        "pa_overlap_hist": (C.c_int, [vp, vp]),
        "pa_overlap_hist_static": (C.c_int, [vp, C.c_int32, C.c_int64, vp, C.c_int, vp]),
        "pa_static_last_error": (C.c_char_p, []),
        "pa_dist_init": (C.c_int, [C.POINTER(PaConfig), C.c_int32, C.c_int32, C.POINTER(vp)]),
        "pa_dist_workspace_bytes": (C.c_uint64, [C.POINTER(PaConfig), C.c_int32]),
        "pa_dist_begin": (C.c_int, [vp, C.c_double, C.c_int32, C.POINTER(PaDistPartial)]),
        "pa_dist_resample": (C.c_int, [vp, C.POINTER(PaDistPartial), i64p]),
        "pa_dist_exchange_plan": (C.c_int, [C.c_int32, i64p, C.c_int32, C.c_uint32, C.c_uint32, i64p, i64p, i64p]),
        "pa_dist_plan_check": (C.c_int, [C.c_int32, i64p, i64p, i64p, i64p]),
        "pa_dist_pack": (C.c_int, [vp, i64p, i32p]),
        "pa_dist_capacity": (C.c_int, [vp, i64p]),
        "pa_dist_buffers": (C.c_int, [vp, C.POINTER(vp), C.POINTER(vp)]),
        "pa_dist_finish": (C.c_int, [vp, i64p, C.POINTER(PaObs)]),
        "pa_dist_new_count": (C.c_int, [vp, i64p, i64p, i64p]),
        "pa_dist_abort": (C.c_int, [vp]),
        "pa_profile_read": (C.c_int, [vp, f64p, i64p]),
        "pa_launch_count": (C.c_int, [vp, i64p]),
        "pa_last_error": (C.c_char_p, [vp]),
        "pa_destroy": (C.c_int, [vp]),
    }
    for name, (res, args) in proto.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _np_ptr(a):
    return C.c_void_p(a.ctypes.data)


def exchange_plan(T, policy=PA_POLICY_BALANCED, block=0, maxexc=0):
    """pa_dist_exchange_plan (pure host function; works without a GPU): T = offspring totals in rank order.
    Returns (new_start[world+1], base[world+1], counts[world, world]) with counts[src, dst] = children src sends to dst;
    raises PaError(PA_EEXTINCT) for an extinct population, PaError(PA_ECAPACITY) if a rank reported -1."""
    lib = load_library()
    t = np.ascontiguousarray(T, np.int64)
    W = t.shape[0]
    ns, base, counts = np.zeros(W + 1, np.int64), np.zeros(W + 1, np.int64), np.zeros((W, W), np.int64)
    p64 = lambda a: a.ctypes.data_as(C.POINTER(C.c_int64))
    rc = lib.pa_dist_exchange_plan(W, p64(t), int(policy), int(block), int(maxexc), p64(ns), p64(base), p64(counts))
    if rc != PA_OK:
        raise PaError(rc, {PA_EEXTINCT: "population extinct", PA_ECAPACITY: "a rank's offspring exceed its capacity"}.get(rc, "bad plan arguments"))
    return ns, base, counts


def overlap_hist_static(spins, L, R=None, out=None, stream=None):
    """pa_overlap_hist_static: the overlap histogram of lattices the caller holds, for callers that cannot allocate
    (no context, no workspace; the library's built-in scratch array holds the bins, L <= 128).

    spins: torch uint8/int32 tensor on the current CUDA device holding R packed lattices (layout C2), R defaults to
    what the tensor holds.  out: None -> a new numpy uint64 array of L*L + 1 entries is returned (the call has then
    synchronised the stream); a torch int64 CUDA tensor of L*L + 1 entries -> filled asynchronously on `stream` and
    returned.  stream: torch stream (default: the current one).  Calls that can overlap on the GPU race on the scratch."""
    import torch
    lib = load_library()
    L = int(L)
    N = L * L
    nbytes = spins.numel() * spins.element_size()
    R = nbytes // max(N // 8, 1) if R is None else int(R)
    if R * (N // 8) > nbytes:
        raise PaError(PA_EINVAL, "overlap_hist_static: the tensor holds fewer than R lattices")
    st = torch.cuda.current_stream(spins.device) if stream is None else stream
    if out is None:
        h = np.zeros(N + 1, np.uint64)
        dst, on_dev = _np_ptr(h), 0
    else:
        if out.numel() * out.element_size() < (N + 1) * 8 or not out.is_cuda:
            raise PaError(PA_EINVAL, "overlap_hist_static: out must be a CUDA tensor of L*L + 1 64-bit entries")
        h, dst, on_dev = out, C.c_void_p(out.data_ptr()), 1
    rc = lib.pa_overlap_hist_static(C.c_void_p(spins.data_ptr()), L, R, dst, on_dev, C.c_void_p(st.cuda_stream))
    if rc != PA_OK:
        raise PaError(rc, lib.pa_static_last_error().decode())
    return h


def plan_check(new_start, caps=None, base=None, R_cur=None):
    """pa_dist_plan_check (pure host function): raises PaError(PA_ECAPACITY) if some rank's new share exceeds that rank's
    capacity, PaError(PA_EEXTINCT) if some rank's new share is empty.  Same verdict on every rank (same inputs).  base
    (from exchange_plan) and R_cur (current populations in rank order): the step has theta > 0 and lands what a rank
    receives behind its parents."""
    lib = load_library()
    ns = np.ascontiguousarray(new_start, np.int64)
    W = ns.shape[0] - 1
    p64 = lambda a: a.ctypes.data_as(C.POINTER(C.c_int64)) if a is not None else None
    arrs = []
    for a, n in ((caps, W), (base, W + 1), (R_cur, W)):
        if a is not None:
            a = np.ascontiguousarray(a, np.int64)
            if a.shape[0] != n:
                raise PaError(PA_EINVAL, "plan_check: array length does not match the number of ranks")
        arrs.append(a)
    rc = lib.pa_dist_plan_check(W, p64(ns), p64(arrs[0]), p64(arrs[1]), p64(arrs[2]))
    if rc != PA_OK:
        raise PaError(rc, {PA_ECAPACITY: "a rank's share of the new population exceeds its capacity",
                           PA_EEXTINCT: "a rank's share of the new population is empty"}.get(rc, "bad plan"))


class PopulationAnnealer:
    """One PA context on the current CUDA device.  Method names mirror the C ABI (pa_*)."""

    def __init__(self, L, R0, P=1, seed=0, beta0=0.0, capacity=0, flags=0, device=None, stream=None,
                 policy=PA_POLICY_BALANCED, block=0, maxexc=0, rank=None, world=None):
        """rank / world given: this context is one rank's shard of a multi-GPU run (pa_dist_init; R0 is the GLOBAL
        target population) and is stepped with dist_begin / dist_resample / dist_finish (see dist.ShardedAnnealer)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2006_00561_b200 needs a CUDA device (no CPU fallback)")
        self._lib = load_library()
        self._torch = torch
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = torch.cuda.current_stream(self.device) if stream is None else stream
        self.L, self.N, self.P, self.R0, self.seed = int(L), int(L) * int(L), int(P), int(R0), int(seed)
        self.wpr = self.N // 32
        cfg = PaConfig(L=L, P=P, R0=R0, capacity=capacity, seed=seed, beta0=beta0, workspace=None, workspace_bytes=0,
                       stream=self.stream.cuda_stream, flags=flags, policy=policy, block=block, maxexc=maxexc)
        self.rank, self.world = rank, world
        if world is None:
            nbytes = self._lib.pa_workspace_bytes(C.byref(cfg))
        else:
            nbytes = self._lib.pa_dist_workspace_bytes(C.byref(cfg), int(world))
        if nbytes == 0:
            raise PaError(PA_EINVAL, "invalid configuration")
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        aligned = (base + 255) // 256 * 256
        cfg.workspace = aligned
        cfg.workspace_bytes = nbytes
        self.workspace_bytes = nbytes
        self._ctx = C.c_void_p()
        if world is None:
            rc = self._lib.pa_init(C.byref(cfg), C.byref(self._ctx))
        else:
            rc = self._lib.pa_dist_init(C.byref(cfg), int(rank), int(world), C.byref(self._ctx))
        if rc != PA_OK:
            msg = self._lib.pa_last_error(self._ctx).decode() if self._ctx else "pa_init failed"
            if self._ctx:
                self._lib.pa_destroy(self._ctx)
                self._ctx = None
            raise PaError(rc, msg)

    # ---- helpers ---------------------------------------------------------------------------------
    def _check(self, rc):
        if rc != PA_OK:
            raise PaError(rc, self._lib.pa_last_error(self._ctx).decode())

    def close(self):
        if getattr(self, "_ctx", None):
            self._lib.pa_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the path --------------------------------------------------------------------------------
    def step(self, beta_next, theta):
        self._check(self._lib.pa_step(self._ctx, float(beta_next), int(theta)))

    def adaptive_beta(self, target_overlap, dbeta_max):
        b = C.c_double(0)
        self._check(self._lib.pa_adaptive_beta(self._ctx, float(target_overlap), float(dbeta_max), C.byref(b)))
        return float(b.value)

    def run(self, betas, theta):
        b = np.ascontiguousarray(betas, np.float64)
        done = C.c_int32(0)
        rc = self._lib.pa_run(self._ctx, b.ctypes.data_as(C.POINTER(C.c_double)), b.shape[0], int(theta), C.byref(done))
        self._check(rc)
        return int(done.value)

    @property
    def R(self):
        r = C.c_int64(0)
        self._check(self._lib.pa_population(self._ctx, C.byref(r)))
        return int(r.value)

    def beta_steps(self):
        b, s = C.c_double(0), C.c_int64(0)
        self._check(self._lib.pa_beta(self._ctx, C.byref(b), C.byref(s)))
        return float(b.value), int(s.value)

    def replica_steps(self):
        r = C.c_int64(0)
        self._check(self._lib.pa_totals(self._ctx, C.byref(r)))
        return int(r.value)

    # host-pointer variants for the end-to-end leg of bench.py (pinned torch CPU tensors)
    def set_spins_host_tensor(self, t, R):
        self._check(self._lib.pa_set_spins(self._ctx, C.c_void_p(t.data_ptr()), int(R), 0))

    def spins_into_host_tensor(self, t, count):
        self._check(self._lib.pa_spins(self._ctx, C.c_void_p(t.data_ptr()), 0, int(count), 0))

    def energies_into_host_tensors(self, tE, tM, n):
        self._check(self._lib.pa_energies(self._ctx, C.c_void_p(tE.data_ptr()), C.c_void_p(tM.data_ptr()), int(n), 0))

    def counts_device(self):
        """offsets off[0..parents] as a torch int32 tensor on the device (measurement helper)"""
        torch = self._torch
        npar = self.parents()
        off = torch.empty(npar + 1, dtype=torch.int32, device=self.device)
        self._check(self._lib.pa_counts(self._ctx, None, C.c_void_p(off.data_ptr()), npar, 1))
        return off

    def energies(self, n=None):
        n = self.R if n is None else int(n)
        E, M = np.empty(n, np.int32), np.empty(n, np.int32)
        self._check(self._lib.pa_energies(self._ctx, _np_ptr(E), _np_ptr(M), n, 0))
        return E, M

    def energies_device(self, n=None):
        torch = self._torch
        n = self.R if n is None else int(n)
        E = torch.empty(n, dtype=torch.int32, device=self.device)
        M = torch.empty(n, dtype=torch.int32, device=self.device)
        self._check(self._lib.pa_energies(self._ctx, C.c_void_p(E.data_ptr()), C.c_void_p(M.data_ptr()), n, 1))
        return E, M

    def log_Z(self):
        a, b, q = C.c_double(0), C.c_double(0), C.c_double(0)
        self._check(self._lib.pa_log_Z(self._ctx, C.byref(a), C.byref(b), C.byref(q)))
        return {"lnZ": float(a.value), "sum_lnQ": float(b.value), "last_Q": float(q.value)}

    def observables(self):
        o = PaObs()
        self._check(self._lib.pa_observables(self._ctx, C.byref(o)))
        big = lambda p: int(p[0]) | (int(p[1]) << 64)
        return {"R": int(o.R), "sum_E": int(o.sum_E), "sum_E2": big(o.sum_E2), "sum_absM": big(o.sum_absM),
                "sum_M2": big(o.sum_M2), "sum_M4": big(o.sum_M4), "mean_E": o.mean_E, "mean_E2": o.mean_E2,
                "mean_absM": o.mean_absM, "mean_M2": o.mean_M2, "mean_M4": o.mean_M4}

    def spins(self, first=0, count=None):
        count = self.R - first if count is None else int(count)
        out = np.empty((count, self.wpr), np.uint32)
        self._check(self._lib.pa_spins(self._ctx, _np_ptr(out), int(first), count, 0))
        return out

    def tau(self, n=None):
        n = self.parents() if n is None else int(n)
        out = np.empty(n, np.float64)
        self._check(self._lib.pa_tau(self._ctx, _np_ptr(out), n, 0))
        return out

    def counts(self, want_n=True):
        npar = self.parents()
        off = np.empty(npar + 1, np.uint32)
        n = np.empty(npar, np.uint32) if want_n else None
        self._check(self._lib.pa_counts(self._ctx, _np_ptr(n) if want_n else None, _np_ptr(off), npar, 0))
        return n, off

    def parents(self):
        r = C.c_int64(0)
        self._check(self._lib.pa_parents(self._ctx, C.byref(r)))
        return int(r.value)

    def partitions(self):
        ps = np.empty(self.P + 1, np.uint32)
        st = np.empty((self.P, 4), np.uint32)
        moved = C.c_int64(0)
        self._check(self._lib.pa_partitions(self._ctx, _np_ptr(ps), _np_ptr(st), C.byref(moved)))
        return ps, st, int(moved.value)

    def thresholds(self):
        a, b = C.c_uint32(0), C.c_uint32(0)
        self._check(self._lib.pa_thresholds(self._ctx, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def set_spins(self, packed):
        if hasattr(packed, "data_ptr"):  # torch tensor on the device
            R = int(packed.shape[0])
            self._check(self._lib.pa_set_spins(self._ctx, C.c_void_p(packed.data_ptr()), R, 1))
        else:
            a = np.ascontiguousarray(packed, np.uint32)
            self._check(self._lib.pa_set_spins(self._ctx, _np_ptr(a), a.shape[0], 0))

    def debug_set_thresholds(self, enable, T4=0, T8=0):
        self._check(self._lib.pa_debug_set_thresholds(self._ctx, int(bool(enable)), int(T4), int(T8)))

    # ---- second Hamiltonian: the 2D +-J spin glass (include/pa_b200.h) --------------------------------
    def set_bonds(self, Jx, Jy):
        """Jx, Jy: the two coupling planes as uint32 words in layout C2 (bit 1 <-> J = +1), N/32 words each; or
        both None for the ferromagnet.  Only before the first step."""
        if Jx is None and Jy is None:
            self._check(self._lib.pa_set_bonds(self._ctx, None, None))
            return
        a = np.ascontiguousarray(Jx, np.uint32).reshape(-1)
        b = np.ascontiguousarray(Jy, np.uint32).reshape(-1)
        if a.shape[0] != self.wpr or b.shape[0] != self.wpr:
            raise PaError(PA_EINVAL, "set_bonds: each coupling plane has N/32 words")
        self._check(self._lib.pa_set_bonds(self._ctx, _np_ptr(a), _np_ptr(b)))

    def overlap_hist(self):
        """hist[(q + N) / 2] over the replica pairs (j, j + R // 2)"""
        h = np.zeros(self.N + 1, np.uint64)
        self._check(self._lib.pa_overlap_hist(self._ctx, _np_ptr(h)))
        return h

    # ---- multi-GPU shard (include/pa_b200.h "multi-GPU") --------------------------------------------
    def dist_begin(self, beta_next, theta):
        p = PaDistPartial()
        self._check(self._lib.pa_dist_begin(self._ctx, float(beta_next), int(theta), C.byref(p)))
        return float(p.sumw), int(p.R)

    def dist_resample(self, partials):
        arr = (PaDistPartial * len(partials))(*[PaDistPartial(float(a), int(b)) for a, b in partials])
        T = C.c_int64(0)
        self._check(self._lib.pa_dist_resample(self._ctx, arr, C.byref(T)))
        return int(T.value)

    def dist_capacity(self):
        r = C.c_int64(0)
        self._check(self._lib.pa_dist_capacity(self._ctx, C.byref(r)))
        return int(r.value)

    def dist_pack(self, T_all):
        """pa_dist_pack; returns True when the rank's own share travels through the exchange buffers (theta = 0)"""
        t = np.ascontiguousarray(T_all, np.int64)
        f = C.c_int32(1)
        self._check(self._lib.pa_dist_pack(self._ctx, t.ctypes.data_as(C.POINTER(C.c_int64)), C.byref(f)))
        return bool(f.value)

    def dist_buffers(self):
        """(children, population) as uint8 views of the workspace tensor: send side / receive side of the exchange"""
        a, b = C.c_void_p(), C.c_void_p()
        self._check(self._lib.pa_dist_buffers(self._ctx, C.byref(a), C.byref(b)))
        base = self.workspace.data_ptr()
        return self.workspace[a.value - base:], self.workspace[b.value - base:]

    def dist_new_count(self, T_all):
        t = np.ascontiguousarray(T_all, np.int64)
        n, first = C.c_int64(0), C.c_int64(0)
        self._check(self._lib.pa_dist_new_count(self._ctx, t.ctypes.data_as(C.POINTER(C.c_int64)), C.byref(n), C.byref(first)))
        return int(n.value), int(first.value)

    def dist_finish(self, T_all):
        t = np.ascontiguousarray(T_all, np.int64)
        o = PaObs()
        self._check(self._lib.pa_dist_finish(self._ctx, t.ctypes.data_as(C.POINTER(C.c_int64)), C.byref(o)))
        big = lambda p: int(p[0]) | (int(p[1]) << 64)
        return {"R": int(o.R), "sum_E": int(o.sum_E), "sum_E2": big(o.sum_E2), "sum_absM": big(o.sum_absM),
                "sum_M2": big(o.sum_M2), "sum_M4": big(o.sum_M4)}

    def dist_abort(self):
        self._check(self._lib.pa_dist_abort(self._ctx))

    def profile_read(self):
        ms = (C.c_double * len(KERNELS))()
        cnt = (C.c_int64 * len(KERNELS))()
        self._check(self._lib.pa_profile_read(self._ctx, ms, cnt))
        return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(KERNELS)}

    def launch_count(self):
        r = C.c_int64(0)
        self._check(self._lib.pa_launch_count(self._ctx, C.byref(r)))
        return int(r.value)
