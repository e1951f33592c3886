"""ctypes wrapper around liboracle.so (TEST INFRASTRUCTURE ONLY, see oracle/__init__.py).

A simulation is described by a plain dict (the same neutral dict the CUDA binding accepts;
neither binding imports the other):

    {"seed": int, "grid": (w, h), "species": [ {"n_loci", "kind": "bit"|"q10", "chrom_len",
      "linkage": "interval"|"poisson", "r", "xover_mean", "mu", "mut_sd", "pheno_scale",
      "fecundity": "bh"|"logistic"|"captures", "fec_a", "K", "K_patch",
      "gaussian": None|{"theta0","dtheta","omega","theta_patch"},
      "predation": None|{"attack","predator"}, "migration", "capacity"} ]}
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# ORACLE_SANITIZE=1: the same source built with AddressSanitizer + UndefinedBehaviorSanitizer into a library of
# its own (profiles/r03_sanitizer.md has the full command, which also needs the two
# sanitizer runtimes in LD_PRELOAD because the host process is python).  Same arithmetic flags otherwise.
_SANITIZE = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")
_SO = os.path.join(_HERE, "liboracle_san.so" if _SANITIZE else "liboracle.so")
_SRC = os.path.join(_HERE, "spegg_oracle.cpp")
TMAX = 128


def build(force=False):
    """Compile the oracle (g++ -O2, fp contraction off).  Building the checker is not using it."""
    hdr = os.path.join(_HERE, "spegg_oracle.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(hdr))):
        return _SO
    cmd = ["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-o", _SO, _SRC]
    if _SANITIZE:
        cmd[1:2] = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


class _SpeciesParams(C.Structure):
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


class _Params(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("n_species", C.c_uint32), ("grid_w", C.c_uint32),
                ("grid_h", C.c_uint32), ("species", C.POINTER(_SpeciesParams))]


class LogEntry(C.Structure):
    _fields_ = [("n_t", C.c_uint64), ("m_t", C.c_uint64), ("n_next", C.c_uint64),
                ("sum_zi", C.c_int64), ("sum_zi2", C.c_int64), ("captures", C.c_uint64),
                ("near_ties", C.c_uint64), ("flags", C.c_uint32), ("step", C.c_uint32)]


class _DebugView(C.Structure):
    _fields_ = [
        ("n_t", C.c_uint64), ("m_t", C.c_uint64), ("f", C.POINTER(C.c_uint8)),
        ("off", C.POINTER(C.c_uint32)), ("mother", C.POINTER(C.c_uint32)),
        ("father", C.POINTER(C.c_uint32)), ("dest", C.POINTER(C.c_uint32)),
        ("u01", C.POINTER(C.c_float)), ("s", C.POINTER(C.c_float)), ("z", C.POINTER(C.c_float)),
        ("zi", C.POINTER(C.c_int32)), ("alive", C.POINTER(C.c_uint8)),
        ("captured", C.POINTER(C.c_uint8)), ("offspring", C.c_void_p),
        ("tables", C.POINTER(C.c_uint32)), ("table_len", C.POINTER(C.c_uint32)),
        ("n_tables", C.c_uint32), ("theta_t", C.c_float), ("zbar_pred", C.c_float),
        ("attack_n", C.c_float), ("cap", C.POINTER(C.c_uint32)),
        ("a_alive", C.POINTER(C.c_uint8)), ("a_u", C.POINTER(C.c_float)), ("a_s", C.POINTER(C.c_float)),
        ("mate_cum", C.POINTER(C.c_uint64)), ("zbar_self", C.c_float),
        ("sex_off", C.POINTER(C.c_uint8)), ("mom_cum", C.POINTER(C.c_uint64)),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Params)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_write_state.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64, C.c_void_p, C.c_void_p, C.c_uint32]
        L.orc_step.argtypes = [C.c_void_p, C.c_uint32]
        L.orc_write_sex.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64, C.c_void_p]
        L.orc_read_sex.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p]
        L.orc_n.restype = C.c_uint64
        L.orc_n.argtypes = [C.c_void_p, C.c_uint32]
        L.orc_step_counter.restype = C.c_uint32
        L.orc_step_counter.argtypes = [C.c_void_p]
        L.orc_flags.restype = C.c_uint32
        L.orc_flags.argtypes = [C.c_void_p]
        L.orc_read_state.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_log_len.restype = C.c_uint32
        L.orc_log_len.argtypes = [C.c_void_p, C.c_uint32]
        L.orc_read_log.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32, C.POINTER(LogEntry)]
        L.orc_make_gamete.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p]
        L.orc_debug.argtypes = [C.c_void_p, C.c_uint32, C.POINTER(_DebugView)]
        L.orc_exp_neg64.restype = C.c_double
        L.orc_exp_neg64.argtypes = [C.c_double]
        L.orc_expf_spec.restype = C.c_float
        L.orc_expf_spec.argtypes = [C.c_float]
        L.orc_poisson_table.argtypes = [C.c_double, C.c_void_p]
        L.orc_poisson_count.argtypes = [C.c_void_p, C.c_int, C.c_uint32]
        L.orc_normal_table.argtypes = [C.c_double, C.c_void_p, C.c_int]
        L.orc_normal_delta.argtypes = [C.c_void_p, C.c_int, C.c_uint32]
        L.orc_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_draw.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p]
        _lib = L
    return _lib


# ------------------------------------------------------------------ primitives
def philox4x32_10(key, ctr):
    k = np.asarray(key, dtype=np.uint32)
    c = np.asarray(ctr, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(k.ctypes.data, c.ctypes.data, out.ctypes.data)
    return out


def draw(seed, species, stream, entity, block, step):
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_draw(seed, species, stream, entity, block, step, out.ctypes.data)
    return out


def exp_neg64(lam):
    return lib().orc_exp_neg64(float(lam))


def expf_spec(x):
    return lib().orc_expf_spec(float(x))


def poisson_table(lam):
    T = np.zeros(TMAX, dtype=np.uint32)
    n = lib().orc_poisson_table(float(lam), T.ctypes.data)
    return T[:n].copy()


def poisson_count(T, u):
    T = np.ascontiguousarray(T, dtype=np.uint32)
    return lib().orc_poisson_count(T.ctypes.data, len(T), int(u))


def normal_table(sigma_over_q):
    T = np.zeros(8192, dtype=np.uint32)
    R = lib().orc_normal_table(float(sigma_over_q), T.ctypes.data, len(T))
    return R, T[: 2 * R].copy()


def normal_delta(T, R, u):
    T = np.ascontiguousarray(T, dtype=np.uint32)
    return lib().orc_normal_delta(T.ctypes.data, int(R), int(u))


# ------------------------------------------------------------------- simulator
_KIND = {"bit": 0, "q10": 1}
_LINK = {"interval": 0, "poisson": 1}
_FEC = {"bh": 0, "logistic": 1, "captures": 2}


def _ptr(arr, ctype):
    return arr.ctypes.data_as(C.POINTER(ctype))


class Oracle:
    """One oracle simulation.  rows: bit -> uint32 [n, 2*L/32]; q10 -> int16 [n, 2*L]."""

    def __init__(self, cfg):
        self.cfg = cfg
        self._keep = []
        ns = len(cfg["species"])
        arr = (_SpeciesParams * ns)()
        w, h = cfg.get("grid", (1, 1))
        self.P = w * h
        self.row_shape = []
        self.row_dtype = []
        for i, sp in enumerate(cfg["species"]):
            p = arr[i]
            L = int(sp["n_loci"])
            p.n_loci = L
            p.genome_kind = _KIND[sp["kind"]]
            cl = np.asarray(sp["chrom_len"], dtype=np.uint32)
            self._keep.append(cl)
            p.n_chrom = len(cl)
            p.chrom_len = _ptr(cl, C.c_uint32)
            p.linkage_mode = _LINK[sp["linkage"]]
            if sp.get("r") is not None:
                r = np.ascontiguousarray(sp["r"], dtype=np.float64)
                assert len(r) == L - 1
                self._keep.append(r)
                p.r = _ptr(r, C.c_double)
            if sp.get("xover_mean") is not None:
                xm = np.ascontiguousarray(sp["xover_mean"], dtype=np.float64)
                assert len(xm) == len(cl)
                self._keep.append(xm)
                p.xover_mean = _ptr(xm, C.c_double)
            p.mu = sp["mu"]
            p.mut_sd = sp.get("mut_sd", 0.0)
            p.pheno_scale = sp["pheno_scale"]
            p.fecundity_model = _FEC[sp["fecundity"]]
            p.fec_a = sp["fec_a"]
            p.K = sp["K"]
            if sp.get("K_patch") is not None:
                kp = np.ascontiguousarray(sp["K_patch"], dtype=np.float64)
                assert len(kp) == self.P
                self._keep.append(kp)
                p.K_patch = _ptr(kp, C.c_double)
            g = sp.get("gaussian")
            if g is not None:
                p.sel_gaussian = 1
                p.theta0, p.dtheta, p.omega = g["theta0"], g.get("dtheta", 0.0), g["omega"]
                if g.get("theta_patch") is not None:
                    tp = np.ascontiguousarray(g["theta_patch"], dtype=np.float32)
                    assert len(tp) == self.P
                    self._keep.append(tp)
                    p.theta_patch = _ptr(tp, C.c_float)
            pr = sp.get("predation")
            if pr is not None:
                p.sel_predation = 1
                p.attack = pr["attack"]
                p.predator_species = pr["predator"]
                p.encounters = pr.get("encounters", 0)
            p.migration = sp.get("migration", 0.0)
            p.capacity = sp["capacity"]
            p.resid_sd = sp.get("resid_sd", 0.0)
            p.adult_survival = sp.get("adult_survival", 0.0)
            p.mate_skew = sp.get("mate_skew", 0.0)
            p.separate_sexes = 1 if sp.get("separate_sexes") else 0
            p.fec_cost = sp.get("fec_cost", 0.0)
            p.assort = sp.get("assort", 0.0)
            p.mother_skew = sp.get("mother_skew", 0.0)
            p.monogamy = 1 if sp.get("monogamy") else 0
            if sp["kind"] == "bit":
                self.row_shape.append(2 * (L // 32))
                self.row_dtype.append(np.uint32)
            else:
                self.row_shape.append(2 * L)
                self.row_dtype.append(np.int16)
        self._arr = arr
        prm = _Params(cfg["seed"], ns, w, h, arr)
        self._h = lib().orc_create(C.byref(prm))
        if not self._h:
            raise ValueError("oracle rejected the parameters")

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def write_state(self, species, rows, patch_start=None, step=0):
        rows = np.ascontiguousarray(rows, dtype=self.row_dtype[species])
        assert rows.ndim == 2 and rows.shape[1] == self.row_shape[species]
        ps = None
        if patch_start is not None:
            ps = np.ascontiguousarray(patch_start, dtype=np.uint32)
        rc = lib().orc_write_state(self._h, species, rows.shape[0], rows.ctypes.data,
                                   ps.ctypes.data if ps is not None else None, step)
        if rc != 0:
            raise ValueError("orc_write_state failed")

    def write_sex(self, species, sex):
        sex = np.ascontiguousarray(sex, dtype=np.uint8)
        if lib().orc_write_sex(self._h, species, sex.shape[0], sex.ctypes.data) != 0:
            raise ValueError("orc_write_sex failed")

    def read_sex(self, species=0):
        out = np.zeros(self.n(species), dtype=np.uint8)
        lib().orc_read_sex(self._h, species, out.ctypes.data)
        return out

    def step(self, n=1):
        lib().orc_step(self._h, n)

    def n(self, species=0):
        return int(lib().orc_n(self._h, species))

    @property
    def step_counter(self):
        return int(lib().orc_step_counter(self._h))

    @property
    def flags(self):
        return int(lib().orc_flags(self._h))

    def read_state(self, species=0):
        n = self.n(species)
        rows = np.zeros((n, self.row_shape[species]), dtype=self.row_dtype[species])
        ps = np.zeros(self.P + 1, dtype=np.uint32)
        zi = np.zeros(n, dtype=np.int32)
        lib().orc_read_state(self._h, species, rows.ctypes.data, ps.ctypes.data, zi.ctypes.data)
        return rows, ps, zi

    def log(self, species=0):
        n = lib().orc_log_len(self._h, species)
        buf = (LogEntry * n)()
        if n:
            lib().orc_read_log(self._h, species, 0, n, buf)
        return [{f[0]: getattr(e, f[0]) for f in LogEntry._fields_} for e in buf]

    def make_gamete(self, species, parent_row, gamete, entity, step):
        row = np.ascontiguousarray(parent_row, dtype=self.row_dtype[species])
        out = np.zeros(self.row_shape[species] // 2, dtype=self.row_dtype[species])
        lib().orc_make_gamete(self._h, species, row.ctypes.data, gamete, entity, step, out.ctypes.data)
        return out

    def debug(self, species=0):
        """Copies of every intermediate of the last step of `species`."""
        v = _DebugView()
        lib().orc_debug(self._h, species, C.byref(v))
        n, m = int(v.n_t), int(v.m_t)

        def arr(p, cnt, dt):
            if cnt == 0:
                return np.zeros(0, dtype=dt)
            return np.ctypeslib.as_array(p, shape=(cnt,)).astype(dt, copy=True)

        d = {
            "n_t": n, "m_t": m,
            "f": arr(v.f, n, np.uint8), "off": arr(v.off, n, np.uint32),
            "mother": arr(v.mother, m, np.uint32), "father": arr(v.father, m, np.uint32),
            "dest": arr(v.dest, m, np.uint32), "u01": arr(v.u01, m, np.float32),
            "s": arr(v.s, m, np.float32), "z": arr(v.z, m, np.float32),
            "zi": arr(v.zi, m, np.int32), "alive": arr(v.alive, m, np.uint8),
            "captured": arr(v.captured, m, np.uint8),
            "a_alive": arr(v.a_alive, n, np.uint8), "a_u": arr(v.a_u, n, np.float32), "a_s": arr(v.a_s, n, np.float32),
            "theta_t": float(v.theta_t), "zbar_pred": float(v.zbar_pred), "attack_n": float(v.attack_n),
            "zbar_self": float(v.zbar_self),
            "mate_cum": (arr(v.mate_cum, n, np.uint64)
                         if (self.cfg["species"][species].get("mate_skew", 0.0) != 0.0
                             or self.cfg["species"][species].get("separate_sexes")) else np.zeros(0, np.uint64)),
            "sex_off": arr(v.sex_off, m, np.uint8),
            "mom_cum": (arr(v.mom_cum, n, np.uint64) if self.cfg["species"][species].get("mother_skew", 0.0) != 0.0
                        else np.zeros(0, np.uint64)),
        }
        nt = int(v.n_tables)
        d["table_len"] = arr(v.table_len, nt, np.uint32)
        d["tables"] = arr(v.tables, nt * TMAX, np.uint32).reshape(nt, TMAX) if nt else np.zeros((0, TMAX), np.uint32)
        w = self.row_shape[species]
        dt = self.row_dtype[species]
        if m:
            ct = C.c_uint32 if dt == np.uint32 else C.c_int16
            p = C.cast(v.offspring, C.POINTER(ct))
            d["offspring"] = np.ctypeslib.as_array(p, shape=(m * w,)).astype(dt, copy=True).reshape(m, w)
        else:
            d["offspring"] = np.zeros((0, w), dtype=dt)
        d["cap"] = arr(v.cap, n, np.uint32) if self.cfg["species"][species]["fecundity"] == "captures" else None
        return d
