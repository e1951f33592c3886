"""Thin ctypes binding of libspegg (include/spegg.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch provides the device workspace
(one uint8 tensor) and the stream.  There is no CPU fallback: a missing libspegg.so or a missing
CUDA device raises.  Function names follow the C ABI (spegg_create -> Sim(...), spegg_step ->
Sim.step, ...).  A simulation is described by the same neutral dict as in workloads.py.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libspegg.so")
TMAX = 128

OK, EINVAL, ENOMEM, ECUDA, ERANGE, ESTATE, ELIMIT = 0, -1, -2, -3, -4, -5, -6
STATIC_MAX_N = 4194304   # SPEGG_STATIC_MAX_N of include/spegg.h
FLAG_OVERFLOW, FLAG_EXTINCT = 1, 2


ABI_VERSION = 9   # SPEGG_ABI_VERSION of include/spegg.h


class SpeciesParams(C.Structure):
    _fields_ = [
        ("n_loci", C.c_uint32), ("genome_kind", C.c_uint32), ("n_chrom", C.c_uint32),
        ("chrom_len", C.POINTER(C.c_uint32)), ("linkage_mode", C.c_uint32),
        ("r", C.POINTER(C.c_double)), ("xover_mean", C.POINTER(C.c_double)),
        ("mu", C.c_double), ("mut_sd", C.c_double), ("pheno_scale", C.c_float),
        ("fecundity_model", C.c_uint32), ("fec_a", C.c_double), ("K", C.c_double),
        ("K_patch", C.POINTER(C.c_double)), ("sel_gaussian", C.c_uint32),
        ("theta0", C.c_double), ("dtheta", C.c_double), ("omega", C.c_double),
        ("theta_patch", C.POINTER(C.c_float)), ("sel_predation", C.c_uint32),
        ("attack", C.c_double), ("predator_species", C.c_uint32), ("migration", C.c_double),
        ("capacity", C.c_uint64), ("resid_sd", C.c_double), ("adult_survival", C.c_double),
        ("mate_skew", C.c_double), ("encounters", C.c_uint32), ("separate_sexes", C.c_uint32),
        ("fec_cost", C.c_double), ("assort", C.c_double), ("mother_skew", C.c_double), ("monogamy", C.c_uint32),
    ]


class Params(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("abi_version", C.c_uint32), ("seed", C.c_uint64),
                ("n_species", C.c_uint32), ("grid_w", C.c_uint32), ("grid_h", C.c_uint32),
                ("debug", C.c_uint32), ("log_capacity", C.c_uint32), ("flags", C.c_uint32),
                ("species", C.POINTER(SpeciesParams))]


class LogEntry(C.Structure):
    _fields_ = [("n_t", C.c_uint64), ("m_t", C.c_uint64), ("n_next", C.c_uint64),
                ("sum_zi", C.c_int64), ("sum_zi2", C.c_int64), ("captures", C.c_uint64),
                ("near_ties", C.c_uint64), ("flags", C.c_uint32), ("step", C.c_uint32)]


class DebugView(C.Structure):
    _fields_ = [
        ("n_t", C.c_uint64), ("m_t", C.c_uint64), ("d_f", C.c_void_p), ("d_off", C.c_void_p),
        ("d_mother", C.c_void_p), ("d_father", C.c_void_p), ("d_dest", C.c_void_p),
        ("d_u01", C.c_void_p), ("d_s", C.c_void_p), ("d_zi", C.c_void_p), ("d_alive", C.c_void_p),
        ("d_captured", C.c_void_p), ("d_offspring", C.c_void_p), ("d_tables", C.c_void_p),
        ("d_table_len", C.c_void_p), ("n_tables", C.c_uint32), ("theta_t", C.c_float),
        ("zbar_pred", C.c_float), ("attack_n", C.c_float), ("d_cap", C.c_void_p),
        ("d_a_alive", C.c_void_p), ("d_a_u", C.c_void_p), ("d_a_s", C.c_void_p),
        ("d_mate_cum", C.c_void_p), ("zbar_self", C.c_float), ("d_sex_off", C.c_void_p), ("d_mom_cum", C.c_void_p),
    ]


EXPORTS = ["spegg_workspace_bytes", "spegg_create", "spegg_write_state", "spegg_write_sex", "spegg_read_sex", "spegg_step", "spegg_read_state",
           "spegg_read_log", "spegg_read_debug", "spegg_status", "spegg_launches_per_step",
           "spegg_kernel_timing", "spegg_offsets_static", "spegg_destroy", "spegg_strerror"]

_lib = None


def load():
    """Loads libspegg.so (built in-tree by build.py).  Raises if it is missing: no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise RuntimeError("libspegg.so not built: run `python -m paper_1603_09255_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(_SO)
    vp, u32, u64 = C.c_void_p, C.c_uint32, C.c_uint64
    L.spegg_workspace_bytes.argtypes = [C.POINTER(Params), C.POINTER(u64)]
    L.spegg_create.argtypes = [C.POINTER(Params), vp, u64, vp, C.POINTER(vp)]
    L.spegg_write_state.argtypes = [vp, u32, u64, vp, C.c_int, vp, u32]
    L.spegg_write_sex.argtypes = [vp, u32, u64, vp]
    L.spegg_read_sex.argtypes = [vp, u32, vp, u64]
    L.spegg_step.argtypes = [vp, u32]
    L.spegg_read_state.argtypes = [vp, u32, C.POINTER(u64), C.POINTER(u32), vp, C.c_int, u64, vp, vp]
    L.spegg_read_log.argtypes = [vp, u32, u32, u32, C.POINTER(LogEntry), C.POINTER(u32)]
    L.spegg_read_debug.argtypes = [vp, u32, C.POINTER(DebugView)]
    L.spegg_status.argtypes = [vp, C.POINTER(u32)]
    L.spegg_launches_per_step.argtypes = [vp, C.POINTER(u32)]
    L.spegg_kernel_timing.argtypes = [vp, C.c_int, C.POINTER(C.c_float), C.POINTER(u32)]
    L.spegg_offsets_static.argtypes = [vp, u64, vp, vp, vp]
    L.spegg_destroy.argtypes = [vp]
    L.spegg_destroy.restype = None
    L.spegg_strerror.argtypes = [C.c_int]
    L.spegg_strerror.restype = C.c_char_p
    _lib = L
    return L


class SpeggError(RuntimeError):
    def __init__(self, code):
        self.code = code
        super().__init__("libspegg: %s (%d)" % (load().spegg_strerror(code).decode(), code))


def _check(rc):
    if rc != OK:
        raise SpeggError(rc)


_KIND = {"bit": 0, "q10": 1}
_LINK = {"interval": 0, "poisson": 1}
_FEC = {"bh": 0, "logistic": 1, "captures": 2}


def _ptr(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def make_params(cfg, debug=False, log_capacity=0):
    """dict -> (spegg_params, keepalive list)."""
    keep = []
    ns = len(cfg["species"])
    arr = (SpeciesParams * ns)()
    w, h = cfg.get("grid", (1, 1))
    P = w * h
    for i, sp in enumerate(cfg["species"]):
        p = arr[i]
        L = int(sp["n_loci"])
        p.n_loci, p.genome_kind = L, _KIND[sp["kind"]]
        cl = np.asarray(sp["chrom_len"], dtype=np.uint32)
        keep.append(cl)
        p.n_chrom, p.chrom_len = len(cl), _ptr(cl, C.c_uint32)
        p.linkage_mode = _LINK[sp["linkage"]]
        if sp.get("r") is not None:
            r = np.ascontiguousarray(sp["r"], dtype=np.float64)
            assert len(r) == L - 1
            keep.append(r)
            p.r = _ptr(r, C.c_double)
        if sp.get("xover_mean") is not None:
            xm = np.ascontiguousarray(sp["xover_mean"], dtype=np.float64)
            assert len(xm) == len(cl)
            keep.append(xm)
            p.xover_mean = _ptr(xm, C.c_double)
        p.mu, p.mut_sd, p.pheno_scale = sp["mu"], sp.get("mut_sd", 0.0), sp["pheno_scale"]
        p.resid_sd = sp.get("resid_sd", 0.0)
        p.adult_survival = sp.get("adult_survival", 0.0)
        p.mate_skew = sp.get("mate_skew", 0.0)
        p.separate_sexes = 1 if sp.get("separate_sexes") else 0
        p.fec_cost = sp.get("fec_cost", 0.0)
        p.assort = sp.get("assort", 0.0)
        p.mother_skew = sp.get("mother_skew", 0.0)
        p.monogamy = int(sp.get("monogamy") or 0)
        p.fecundity_model, p.fec_a, p.K = _FEC[sp["fecundity"]], sp["fec_a"], sp["K"]
        if sp.get("K_patch") is not None:
            kp = np.ascontiguousarray(sp["K_patch"], dtype=np.float64)
            assert len(kp) == P
            keep.append(kp)
            p.K_patch = _ptr(kp, C.c_double)
        g = sp.get("gaussian")
        if g is not None:
            p.sel_gaussian = 1
            p.theta0, p.dtheta, p.omega = g["theta0"], g.get("dtheta", 0.0), g["omega"]
            if g.get("theta_patch") is not None:
                tp = np.ascontiguousarray(g["theta_patch"], dtype=np.float32)
                assert len(tp) == P
                keep.append(tp)
                p.theta_patch = _ptr(tp, C.c_float)
        pr = sp.get("predation")
        if pr is not None:
            p.sel_predation, p.attack, p.predator_species = 1, pr["attack"], pr["predator"]
            p.encounters = pr.get("encounters", 0)
        p.migration, p.capacity = sp.get("migration", 0.0), sp["capacity"]
    keep.append(arr)
    prm = Params(C.sizeof(Params), ABI_VERSION, cfg["seed"], ns, w, h, 1 if debug else 0, log_capacity, 0, arr)
    return prm, keep


def workspace_bytes(cfg, debug=False, log_capacity=0):
    prm, keep = make_params(cfg, debug, log_capacity)
    n = C.c_uint64(0)
    _check(load().spegg_workspace_bytes(C.byref(prm), C.byref(n)))
    return int(n.value)


def offsets_static(f, off, total, n=None, stream=None):
    """spegg_offsets_static: neonate offsets of the fecundities `f` without allocating anything.

    For callers that cannot allocate device memory where they stand (see include/spegg.h): the scan's
    scratch is a fixed ~34 KB array inside libspegg.so, so n is limited to STATIC_MAX_N adults and calls
    whose GPU work overlaps on one device race on that array.  f (uint8), off (uint32) and total (one
    int64/uint64 word) are CUDA tensors the caller already owns, on the current device; this wrapper only
    passes their addresses and the stream (default: torch's current stream) -- it creates no tensor.
    The first call on a device resolves the array's address: make it before any stream capture."""
    import torch
    n = f.numel() if n is None else int(n)
    assert f.is_cuda and off.is_cuda and total.is_cuda and f.is_contiguous() and off.is_contiguous()
    assert f.element_size() == 1 and off.element_size() == 4 and total.element_size() == 8
    assert n > STATIC_MAX_N or (n <= f.numel() and n <= off.numel())   # over the limit: the library refuses before it looks at the buffers
    st = torch.cuda.current_stream(f.device).cuda_stream if stream is None else stream
    _check(load().spegg_offsets_static(f.data_ptr() if f.numel() else None, n, off.data_ptr() if off.numel() else None,
                                       total.data_ptr(), st))


class Sim:
    """spegg_sim handle.  rows: bit -> uint32 [n, 2*L/32]; q10 -> int16 [n, 2*L]."""

    def __init__(self, cfg, debug=False, log_capacity=0, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libspegg needs a CUDA device (there is no CPU fallback)")
        self._torch = torch
        self.cfg = cfg
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.lib = load()
        prm, keep = make_params(cfg, debug, log_capacity)
        nbytes = C.c_uint64(0)
        _check(self.lib.spegg_workspace_bytes(C.byref(prm), C.byref(nbytes)))
        self.workspace = torch.empty(int(nbytes.value), dtype=torch.uint8, device=self.device)
        self.stream = torch.cuda.Stream(device=self.device)
        h = C.c_void_p()
        _check(self.lib.spegg_create(C.byref(prm), self.workspace.data_ptr(), nbytes.value,
                                     self.stream.cuda_stream, C.byref(h)))
        self._h = h
        self.debug = debug
        w, hh = cfg.get("grid", (1, 1))
        self.P = w * hh
        self.row_shape, self.row_dtype = [], []
        for sp in cfg["species"]:
            if sp["kind"] == "bit":
                self.row_shape.append(2 * (sp["n_loci"] // 32))
                self.row_dtype.append(np.uint32)
            else:
                self.row_shape.append(2 * sp["n_loci"])
                self.row_dtype.append(np.int16)

    def close(self):
        if getattr(self, "_h", None):
            self.lib.spegg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- spegg_write_state: host numpy rows or a device torch tensor
    def write_state(self, species, rows, patch_start=None, step=0):
        torch = self._torch
        ps = None
        if patch_start is not None:
            ps = np.ascontiguousarray(patch_start, dtype=np.uint32)
        psp = ps.ctypes.data if ps is not None else None
        if isinstance(rows, torch.Tensor):
            assert rows.is_cuda and rows.is_contiguous()
            n = rows.shape[0]
            _check(self.lib.spegg_write_state(self._h, species, n, rows.data_ptr(), 1, psp, step))
        else:
            rows = np.ascontiguousarray(rows, dtype=self.row_dtype[species])
            assert rows.ndim == 2 and rows.shape[1] == self.row_shape[species]
            _check(self.lib.spegg_write_state(self._h, species, rows.shape[0], rows.ctypes.data, 0, psp, step))

    def write_sex(self, species, sex):
        sex = np.ascontiguousarray(sex, dtype=np.uint8)
        _check(self.lib.spegg_write_sex(self._h, species, sex.shape[0], sex.ctypes.data))

    def read_sex(self, species=0):
        out = np.zeros(self.n(species), dtype=np.uint8)
        if len(out):
            _check(self.lib.spegg_read_sex(self._h, species, out.ctypes.data, len(out)))
        return out

    def step(self, n=1):
        _check(self.lib.spegg_step(self._h, n))

    def synchronize(self):
        self.stream.synchronize()

    def n(self, species=0):
        n, st = C.c_uint64(0), C.c_uint32(0)
        _check(self.lib.spegg_read_state(self._h, species, C.byref(n), C.byref(st), None, 0, 0, None, None))
        return int(n.value)

    @property
    def step_counter(self):
        n, st = C.c_uint64(0), C.c_uint32(0)
        _check(self.lib.spegg_read_state(self._h, 0, C.byref(n), C.byref(st), None, 0, 0, None, None))
        return int(st.value)

    def read_state(self, species=0, want_zi=True, out=None):
        """-> (rows, patch_start, zi) as numpy arrays (host copies through the C ABI)."""
        n = self.n(species)
        rows = out if out is not None else np.zeros((n, self.row_shape[species]), dtype=self.row_dtype[species])
        ps = np.zeros(self.P + 1, dtype=np.uint32)
        zi = np.zeros(n, dtype=np.int32) if want_zi else None
        nn, st = C.c_uint64(0), C.c_uint32(0)
        _check(self.lib.spegg_read_state(self._h, species, C.byref(nn), C.byref(st), rows.ctypes.data, 0,
                                         rows.nbytes, ps.ctypes.data, zi.ctypes.data if want_zi else None))
        return rows[:n], ps, zi

    def read_log(self, species=0, last=None):
        """spegg_read_log: all entries written since the last write_state, or only the `last` n of them."""
        avail = C.c_uint32(0)
        _check(self.lib.spegg_read_log(self._h, species, 0, 0, None, C.byref(avail)))
        n = int(avail.value)
        first = 0 if last is None else max(0, n - int(last))
        cnt = n - first
        buf = (LogEntry * max(cnt, 1))()
        if cnt:
            _check(self.lib.spegg_read_log(self._h, species, first, cnt, buf, None))
        return [{f[0]: getattr(buf[i], f[0]) for f in LogEntry._fields_} for i in range(cnt)]

    def status(self):
        f = C.c_uint32(0)
        _check(self.lib.spegg_status(self._h, C.byref(f)))
        return int(f.value)

    def launches_per_step(self):
        n = C.c_uint32(0)
        _check(self.lib.spegg_launches_per_step(self._h, C.byref(n)))
        return int(n.value)

    def kernel_timing(self, enable):
        ms, n = C.c_float(0), C.c_uint32(0)
        _check(self.lib.spegg_kernel_timing(self._h, 1 if enable else 0, C.byref(ms), C.byref(n)))
        return float(ms.value), int(n.value)

    def read_debug(self, species=0):
        """Host copies of every intermediate of the last step (debug=True only)."""
        torch = self._torch
        v = DebugView()
        _check(self.lib.spegg_read_debug(self._h, species, C.byref(v)))
        n, m = int(v.n_t), int(v.m_t)
        base = self.workspace.data_ptr()

        def arr(ptr, cnt, dt):
            if cnt == 0 or not ptr:
                return np.zeros(0, dtype=dt)
            nbytes = cnt * np.dtype(dt).itemsize
            off = ptr - base
            return self.workspace[off:off + nbytes].cpu().numpy().view(dt).copy()

        w, dt = self.row_shape[species], self.row_dtype[species]
        nt = int(v.n_tables)
        d = {
            "n_t": n, "m_t": m,
            "f": arr(v.d_f, n, np.uint8), "off": arr(v.d_off, n, np.uint32),
            "mother": arr(v.d_mother, m, np.uint32), "father": arr(v.d_father, m, np.uint32),
            "dest": arr(v.d_dest, m, np.uint32), "u01": arr(v.d_u01, m, np.float32),
            "s": arr(v.d_s, m, np.float32), "zi": arr(v.d_zi, m, np.int32),
            "alive": arr(v.d_alive, m, np.uint8), "captured": arr(v.d_captured, m, np.uint8),
            "offspring": arr(v.d_offspring, m * w, dt).reshape(m, w),
            "tables": arr(v.d_tables, nt * TMAX, np.uint32).reshape(nt, TMAX),
            "table_len": arr(v.d_table_len, nt, np.uint32),
            "theta_t": float(v.theta_t), "zbar_pred": float(v.zbar_pred), "attack_n": float(v.attack_n),
            "cap": arr(v.d_cap, n, np.uint32),
            "a_alive": arr(v.d_a_alive, n, np.uint8), "a_u": arr(v.d_a_u, n, np.float32),
            "a_s": arr(v.d_a_s, n, np.float32),
            "zbar_self": float(v.zbar_self),
            "mate_cum": (arr(v.d_mate_cum, n, np.uint64)
                         if (self.cfg["species"][species].get("mate_skew", 0.0) != 0.0
                             or self.cfg["species"][species].get("separate_sexes")) else np.zeros(0, np.uint64)),
            "sex_off": (arr(v.d_sex_off, m, np.uint8) if self.cfg["species"][species].get("separate_sexes")
                        else np.zeros(m, np.uint8)),
            "mom_cum": (arr(v.d_mom_cum, n, np.uint64) if self.cfg["species"][species].get("mother_skew", 0.0) != 0.0
                        else np.zeros(0, np.uint64)),
        }
        return d
