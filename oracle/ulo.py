"""ctypes binding of the ORACLE (oracle/ulo.cpp) -- test infrastructure, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It shares nothing with paper_1309_3859_b200/.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libulo.so")
_SRC = [os.path.join(_HERE, "ulo.cpp"), os.path.join(_HERE, "ulo.h")]


def build(force=False):
    """Compile oracle/ulo.cpp with g++ (plain -O2, no fast-math, single thread).  With ULO_SANITIZE=1 in the environment
    the library is the AddressSanitizer + UndefinedBehaviorSanitizer build instead (tests/test_oracle_sanitizers.py; the
    process must then be started with LD_PRELOAD=libasan)."""
    san = os.environ.get("ULO_SANITIZE") == "1"
    so = _SO.replace(".so", "_san.so") if san else _SO
    if not force and os.path.exists(so) and all(os.path.getmtime(so) >= os.path.getmtime(s) for s in _SRC):
        return so
    flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer"] if san else ["-O2"]
    cmd = ["g++", "-std=c++17"] + flags + ["-fPIC", "-shared", "-fno-fast-math", "-ffp-contract=off", "-o", so + ".tmp", _SRC[0]]
    subprocess.run(cmd, check=True, cwd=_HERE)
    os.replace(so + ".tmp", so)
    return so


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        P = C.c_void_p
        L.ulo_create.argtypes = [C.POINTER(P), C.c_int, C.c_int, C.c_double, C.c_uint64]
        L.ulo_destroy.argtypes = [P]
        L.ulo_init.argtypes = [P, C.c_int]
        L.ulo_set_beta.argtypes = [P, C.c_double]
        L.ulo_set_links.argtypes = [P, P]
        L.ulo_get_links.argtypes = [P, P]
        L.ulo_get_counter.argtypes = [P, C.POINTER(C.c_uint64)]
        L.ulo_set_counter.argtypes = [P, C.c_uint64]
        L.ulo_sweep.argtypes = [P, C.c_int, C.c_int]
        L.ulo_substep.argtypes = [P, C.c_int, C.c_int, C.c_int, C.c_int]
        L.ulo_set_subupdate.argtypes = [P, C.c_int, C.c_int, C.c_int]
        L.ulo_set_multihit.argtypes = [P, C.c_int]
        L.ulo_set_update_algorithm.argtypes = [P, C.c_int, C.c_double]
        L.ulo_multilevel.argtypes = [P, C.c_int, C.c_int, C.c_int, P, C.c_int]
        L.ulo_multilevel2.argtypes = [P, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, P, C.c_int]
        L.ulo_measure_begin.argtypes = [P, C.c_int, C.c_int, P, C.c_int]
        L.ulo_accumulate.argtypes = [P]
        L.ulo_measure_end.argtypes = [P]
        L.ulo_measure2_begin.argtypes = [P, C.c_int, C.c_int, C.c_int, P, C.c_int]
        L.ulo_combine.argtypes = [P]
        L.ulo_measure2_end.argtypes = [P]
        L.ulo_read_slab_field_averages.argtypes = [P, P]
        L.ulo_plaquette.argtypes = [P, P]
        L.ulo_read_correlators.argtypes = [P, P, P, P]
        L.ulo_read_slab_averages.argtypes = [P, P]
        L.ulo_last_error.argtypes = [P]
        L.ulo_last_error.restype = C.c_char_p
        L.ulo_philox4x32_10.argtypes = [P, P, P]
        L.ulo_philox4x32_10.restype = None
        L.ulo_staple.argtypes = [P, C.c_int, C.c_long, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.ulo_heatbath_phi.argtypes = [C.c_double, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32,
                                       C.POINTER(C.c_double), C.POINTER(C.c_int)]
        L.ulo_polyakov_naive.argtypes = [P, C.c_int, P, P]
        L.ulo_polyakov.argtypes = [P, C.c_int, P]
        L.ulo_paper_accumulator_bytes.argtypes = [C.c_int, C.c_int, C.c_int]
        L.ulo_paper_accumulator_bytes.restype = C.c_double
    return _lib


class OracleError(RuntimeError):
    pass


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _fps(field_points):
    fp = np.ascontiguousarray(np.asarray(field_points if field_points is not None else [], dtype=np.int32).reshape(-1, 3))
    return fp, fp.shape[0]


class Oracle:
    """Thin object wrapper: one method per ulo_* call, argument marshalling only."""

    def __init__(self, Ns, Nt, beta, seed):
        self.Ns, self.Nt = int(Ns), int(Nt)
        self.V = self.Ns ** 3 * self.Nt
        self._h = C.c_void_p()
        rc = lib().ulo_create(C.byref(self._h), Ns, Nt, float(beta), int(seed))
        if rc != 0:
            self._h = None
            raise OracleError(f"ulo_create failed: {rc}")
        self._meas = None

    def _ck(self, rc):
        if rc != 0:
            raise OracleError(f"oracle error {rc}: {lib().ulo_last_error(self._h).decode()}")

    def close(self):
        if self._h:
            lib().ulo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init(self, mode):
        self._ck(lib().ulo_init(self._h, int(mode)))

    def set_beta(self, beta):
        self._ck(lib().ulo_set_beta(self._h, float(beta)))

    def set_links(self, links):
        a = np.ascontiguousarray(links, dtype=np.float32).reshape(-1)
        assert a.size == 4 * self.V
        self._ck(lib().ulo_set_links(self._h, _ptr(a)))

    def get_links(self):
        a = np.empty((4, self.Nt, self.Ns, self.Ns, self.Ns), dtype=np.float32)
        self._ck(lib().ulo_get_links(self._h, _ptr(a)))
        return a

    def get_counter(self):
        v = C.c_uint64()
        self._ck(lib().ulo_get_counter(self._h, C.byref(v)))
        return v.value

    def set_counter(self, v):
        self._ck(lib().ulo_set_counter(self._h, int(v)))

    def sweep(self, n_hb, n_or):
        self._ck(lib().ulo_sweep(self._h, int(n_hb), int(n_or)))

    def substep(self, kind, parity, mu, slab_d=0):
        self._ck(lib().ulo_substep(self._h, int(kind), int(parity), int(mu), int(slab_d)))

    def set_update_algorithm(self, alg, delta=np.pi):
        self._ck(lib().ulo_set_update_algorithm(self._h, int(alg), float(delta)))

    def set_multihit(self, on):
        self._ck(lib().ulo_set_multihit(self._h, int(on)))

    def set_subupdate(self, n_hb, n_or, k_sweeps=1):
        self._ck(lib().ulo_set_subupdate(self._h, int(n_hb), int(n_or), int(k_sweeps)))

    def multilevel(self, slab_thickness, n_sub, r_max, field_points=None):
        fp, n = _fps(field_points)
        self._ck(lib().ulo_multilevel(self._h, int(slab_thickness), int(n_sub), int(r_max), _ptr(fp), n))
        self._meas = (int(r_max), n, self.Nt // int(slab_thickness))

    def multilevel2(self, d_in, n_in, d_out, n_out, r_max, field_points=None):
        fp, n = _fps(field_points)
        self._ck(lib().ulo_multilevel2(self._h, int(d_in), int(n_in), int(d_out), int(n_out), int(r_max), _ptr(fp), n))
        self._meas = (int(r_max), n, self.Nt // int(d_out))

    def measure_begin(self, slab_thickness, r_max, field_points=None):
        fp, n = _fps(field_points)
        self._ck(lib().ulo_measure_begin(self._h, int(slab_thickness), int(r_max), _ptr(fp), n))
        self._meas = (int(r_max), n, self.Nt // int(slab_thickness))

    def accumulate(self):
        self._ck(lib().ulo_accumulate(self._h))

    def measure_end(self):
        self._ck(lib().ulo_measure_end(self._h))

    def measure2_begin(self, d_in, d_out, r_max, field_points=None):
        fp, n = _fps(field_points)
        self._ck(lib().ulo_measure2_begin(self._h, int(d_in), int(d_out), int(r_max), _ptr(fp), n))
        self._meas = (int(r_max), n, self.Nt // int(d_out))

    def combine(self):
        self._ck(lib().ulo_combine(self._h))

    def measure2_end(self):
        self._ck(lib().ulo_measure2_end(self._h))

    def read_slab_field_averages(self):
        R, F, S = self._meas
        out = np.zeros((3, R, S, F, 12, self.Ns ** 3, 2))
        self._ck(lib().ulo_read_slab_field_averages(self._h, _ptr(out)))
        return out[..., 0] + 1j * out[..., 1]

    def plaquette(self):
        out = np.zeros(3)
        self._ck(lib().ulo_plaquette(self._h, _ptr(out)))
        return out

    def read_correlators(self):
        if self._meas is None:
            self._ck(lib().ulo_read_correlators(self._h, None, None, None))
        R, F, _ = self._meas
        corr = np.zeros((R, 2))
        field = np.zeros((R, max(F, 1), 12, 2))
        vac = np.zeros(12)
        self._ck(lib().ulo_read_correlators(self._h, _ptr(corr), _ptr(field) if F else None, _ptr(vac)))
        return corr[:, 0] + 1j * corr[:, 1], (field[..., 0] + 1j * field[..., 1])[:, :F], vac

    def read_slab_averages(self):
        R, _, S = self._meas
        out = np.zeros((3, R, S, self.Ns ** 3, 2))
        self._ck(lib().ulo_read_slab_averages(self._h, _ptr(out)))
        return out[..., 0] + 1j * out[..., 1]

    def staple(self, mu, site):
        k, a = C.c_double(), C.c_double()
        self._ck(lib().ulo_staple(self._h, int(mu), int(site), C.byref(k), C.byref(a)))
        return k.value, a.value

    def polyakov(self, multihit=0):
        out = np.zeros(2)
        self._ck(lib().ulo_polyakov(self._h, int(multihit), _ptr(out)))
        return complex(out[0], out[1])

    def polyakov_naive(self, r_max):
        corr = np.zeros((max(r_max, 1), 2))
        mp = np.zeros(2)
        self._ck(lib().ulo_polyakov_naive(self._h, int(r_max), _ptr(corr), _ptr(mp)))
        return (corr[:, 0] + 1j * corr[:, 1])[:r_max], complex(mp[0], mp[1])


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().ulo_philox4x32_10(_ptr(c), _ptr(k), _ptr(out))
    return out


def heatbath_phi(a, seed, c0, c1=0, c2=0, c3low=0):
    phi, n = C.c_double(), C.c_int()
    rc = lib().ulo_heatbath_phi(float(a), int(seed), int(c0), int(c1), int(c2), int(c3low), C.byref(phi), C.byref(n))
    if rc != 0:
        raise OracleError(f"ulo_heatbath_phi failed: {rc}")
    return phi.value, n.value


def paper_accumulator_bytes(Ns, Nt, step):
    return lib().ulo_paper_accumulator_bytes(int(Ns), int(Nt), int(step))
