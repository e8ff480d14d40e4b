"""ctypes binding of libul.so -- same names as include/ul.h, argument marshalling only.

PyTorch supplies device memory (``torch.empty`` on ``cuda``) and the stream; every step of the
hot path runs in the library's CUDA kernels.  There is no CPU fallback: if ``libul.so`` is
missing or no CUDA device is present the calls raise.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(_HERE, "libul.so")

UL_OK, UL_EINVAL, UL_ENOMEM, UL_ECUDA, UL_ESTATE = 0, -1, -2, -3, -4

# every symbol include/ul.h declares (tests check that the library exports exactly these)
SYMBOLS = [
    "ul_create", "ul_create_ext", "ul_workspace_bytes", "ul_destroy", "ul_init", "ul_set_beta",
    "ul_set_links", "ul_get_links", "ul_get_links_async", "ul_get_links_wait", "ul_set_links_async", "ul_set_links_commit", "ul_set_links_raw", "ul_get_links_raw", "ul_get_counter", "ul_set_counter", "ul_sweep", "ul_substep", "ul_substep_slabs", "ul_set_slab_group", "ul_set_slab_group_streams",
    "ul_set_subupdate", "ul_set_update_algorithm", "ul_multilevel", "ul_multilevel_replay", "ul_workspace_bytes_replay", "ul_multilevel2_replay", "ul_workspace_bytes_replay2", "ul_multilevel2", "ul_measure_begin", "ul_accumulate",
    "ul_measure_end", "ul_measure2_begin", "ul_combine", "ul_measure2_end", "ul_set_accum_batch", "ul_set_multihit", "ul_plaquette", "ul_plaquette_noalloc", "ul_polyakov", "ul_set_site_offset", "ul_slab_partial_product", "ul_combine_partial_products", "ul_set_halo_peers", "ul_halo_flags", "ul_set_halo_peer_flags", "ul_ipc_export", "ul_ipc_open", "ul_read_correlators", "ul_read_slab_averages",
    "ul_get_launch_count", "ul_philox_selftest", "ul_sync", "ul_last_error",
]

_lib = None


class UlError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libul error {code}: {msg}")
        self.code = code


def lib():
    """Loads libul.so (built by ``python -m paper_1309_3859_b200.build``).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(SO_PATH):
            raise FileNotFoundError(f"{SO_PATH} not built: run `python -m paper_1309_3859_b200.build` "
                                    "(there is no CPU fallback)")
        L = C.CDLL(SO_PATH)
        P = C.c_void_p
        L.ul_create.argtypes = [C.POINTER(P), C.c_int, C.c_int, C.c_double, C.c_uint64]
        L.ul_create_ext.argtypes = [C.POINTER(P), C.c_int, C.c_int, C.c_double, C.c_uint64,
                                    P, C.c_size_t, P, C.c_size_t, P]
        L.ul_workspace_bytes.argtypes = [C.c_int] * 6
        L.ul_workspace_bytes.restype = C.c_size_t
        L.ul_destroy.argtypes = [P]
        L.ul_init.argtypes = [P, C.c_int]
        L.ul_set_beta.argtypes = [P, C.c_double]
        L.ul_set_links.argtypes = [P, P]
        L.ul_get_links.argtypes = [P, P]
        L.ul_get_links_async.argtypes = [P, P]
        L.ul_get_links_wait.argtypes = [P]
        L.ul_set_links_async.argtypes = [P, P]
        L.ul_set_links_commit.argtypes = [P]
        L.ul_set_links_raw.argtypes = [P, P]
        L.ul_get_links_raw.argtypes = [P, P]
        L.ul_get_counter.argtypes = [P, C.POINTER(C.c_uint64)]
        L.ul_set_counter.argtypes = [P, C.c_uint64]
        L.ul_sweep.argtypes = [P, C.c_int, C.c_int]
        L.ul_substep.argtypes = [P, C.c_int, C.c_int, C.c_int, C.c_int]
        L.ul_substep_slabs.argtypes = [P] + [C.c_int] * 6
        L.ul_set_slab_group.argtypes = [P, C.c_int]
        L.ul_set_slab_group_streams.argtypes = [P, C.c_int]
        L.ul_set_subupdate.argtypes = [P, C.c_int, C.c_int, C.c_int]
        L.ul_set_update_algorithm.argtypes = [P, C.c_int, C.c_double]
        L.ul_multilevel.argtypes = [P, C.c_int, C.c_int, C.c_int, P, C.c_int]
        L.ul_multilevel2.argtypes = [P, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, P, C.c_int]
        L.ul_multilevel_replay.argtypes = [P, C.c_int, C.c_int, C.c_int, P, C.c_int]
        L.ul_workspace_bytes_replay.argtypes = [C.c_int] * 5
        L.ul_workspace_bytes_replay.restype = C.c_size_t
        L.ul_multilevel2_replay.argtypes = [P, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, P, C.c_int]
        L.ul_workspace_bytes_replay2.argtypes = [C.c_int] * 6
        L.ul_workspace_bytes_replay2.restype = C.c_size_t
        L.ul_measure_begin.argtypes = [P, C.c_int, C.c_int, P, C.c_int]
        L.ul_set_accum_batch.argtypes = [P, C.c_int]
        L.ul_set_multihit.argtypes = [P, C.c_int]
        L.ul_polyakov.argtypes = [P, C.c_int, P]
        L.ul_set_site_offset.argtypes = [P, C.c_int64]
        L.ul_slab_partial_product.argtypes = [P, C.c_int, C.c_int, P]
        L.ul_combine_partial_products.argtypes = [P, P, C.c_int, P]
        L.ul_set_halo_peers.argtypes = [P, P, P, C.c_int]
        L.ul_halo_flags.argtypes = [P, C.POINTER(P)]
        L.ul_set_halo_peer_flags.argtypes = [P, P, P]
        L.ul_ipc_export.argtypes = [P, P, C.POINTER(C.c_uint64), P, C.POINTER(C.c_uint64)]
        L.ul_ipc_open.argtypes = [P, P, C.c_uint64, C.POINTER(P)]
        L.ul_accumulate.argtypes = [P]
        L.ul_measure_end.argtypes = [P]
        L.ul_measure2_begin.argtypes = [P, C.c_int, C.c_int, C.c_int, P, C.c_int]
        L.ul_combine.argtypes = [P]
        L.ul_measure2_end.argtypes = [P]
        L.ul_plaquette.argtypes = [P, P]
        L.ul_plaquette_noalloc.argtypes = [P, P]
        L.ul_read_correlators.argtypes = [P, P, P, P]
        L.ul_read_slab_averages.argtypes = [P, P]
        L.ul_get_launch_count.argtypes = [P, C.POINTER(C.c_uint64)]
        L.ul_philox_selftest.argtypes = [P, P, P, C.c_int]
        L.ul_sync.argtypes = [P]
        L.ul_last_error.argtypes = [P]
        L.ul_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _fps(field_points):
    fp = np.ascontiguousarray(np.asarray(field_points if field_points is not None else [], dtype=np.int32).reshape(-1, 3))
    return fp, fp.shape[0]


def workspace_bytes(Ns, Nt, d_in, d_out, r_max, n_fp):
    return int(lib().ul_workspace_bytes(int(Ns), int(Nt), int(d_in), int(d_out), int(r_max), int(n_fp)))


def workspace_bytes_replay(Ns, Nt, d, r_max, n_fp):
    return int(lib().ul_workspace_bytes_replay(int(Ns), int(Nt), int(d), int(r_max), int(n_fp)))


def workspace_bytes_replay2(Ns, Nt, d_in, d_out, r_max, n_fp):
    return int(lib().ul_workspace_bytes_replay2(int(Ns), int(Nt), int(d_in), int(d_out), int(r_max), int(n_fp)))


def philox_selftest(ctr, key):
    c = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    k = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    out = np.zeros_like(c)
    rc = lib().ul_philox_selftest(_ptr(c), _ptr(k), _ptr(out), c.shape[0])
    if rc != 0:
        raise UlError(rc, lib().ul_last_error(None).decode())
    return out


class Lattice:
    """One ul_ctx.  Device memory for the links (and, if ``workspace_bytes`` > 0, for the
    multilevel accumulators) comes from torch; kernels run on ``stream`` (a torch.cuda.Stream;
    default: torch's current stream)."""

    def __init__(self, Ns, Nt, beta, seed, workspace_bytes=0, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise UlError(UL_ECUDA, "no CUDA device (there is no CPU fallback)")
        self.Ns, self.Nt = int(Ns), int(Nt)
        self.V = self.Ns ** 3 * self.Nt
        self._torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.links = torch.empty(4 * self.V, dtype=torch.float32, device=self.device)
        self.work = torch.empty(int(workspace_bytes), dtype=torch.uint8, device=self.device) if workspace_bytes else None
        self._h = C.c_void_p()
        rc = lib().ul_create_ext(C.byref(self._h), self.Ns, self.Nt, float(beta), int(seed),
                                 C.c_void_p(self.links.data_ptr()), self.links.numel() * 4,
                                 C.c_void_p(self.work.data_ptr()) if self.work is not None else None,
                                 self.work.numel() if self.work is not None else 0,
                                 C.c_void_p(self.stream.cuda_stream))
        if rc != 0:
            self._h = None
            raise UlError(rc, lib().ul_last_error(None).decode())
        self._meas = None

    def _ck(self, rc):
        if rc != 0:
            raise UlError(rc, lib().ul_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            lib().ul_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init(self, mode):
        self._ck(lib().ul_init(self._h, int(mode)))

    def set_beta(self, beta):
        self._ck(lib().ul_set_beta(self._h, float(beta)))

    def set_links(self, links):
        """links: canonical host array float32[4][Nt][Ns][Ns][Ns] (numpy, or a CPU torch tensor)."""
        if hasattr(links, "data_ptr"):
            assert links.device.type == "cpu" and links.is_contiguous() and links.numel() == 4 * self.V
            self._ck(lib().ul_set_links(self._h, C.c_void_p(links.data_ptr())))
            return
        a = np.ascontiguousarray(links, dtype=np.float32).reshape(-1)
        assert a.size == 4 * self.V
        self._ck(lib().ul_set_links(self._h, _ptr(a)))

    def get_links(self, out=None):
        if out is not None and hasattr(out, "data_ptr"):
            assert out.device.type == "cpu" and out.is_contiguous() and out.numel() == 4 * self.V
            self._ck(lib().ul_get_links(self._h, C.c_void_p(out.data_ptr())))
            return out
        a = np.empty((4, self.Nt, self.Ns, self.Ns, self.Ns), dtype=np.float32) if out is None else out
        self._ck(lib().ul_get_links(self._h, _ptr(a)))
        return a

    def get_links_async(self, out):
        """out: contiguous CPU float32 tensor of 4 V elements (pinned); valid after get_links_wait()."""
        assert out.device.type == "cpu" and out.is_contiguous() and out.numel() == 4 * self.V
        self._ck(lib().ul_get_links_async(self._h, C.c_void_p(out.data_ptr())))
        return out

    def get_links_wait(self):
        self._ck(lib().ul_get_links_wait(self._h))

    def set_links_async(self, src):
        """src: contiguous CPU float32 tensor of 4 V elements (pinned), untouched until set_links_commit() returns."""
        assert src.device.type == "cpu" and src.is_contiguous() and src.numel() == 4 * self.V
        self._ck(lib().ul_set_links_async(self._h, C.c_void_p(src.data_ptr())))

    def set_links_commit(self):
        self._ck(lib().ul_set_links_commit(self._h))

    def set_links_raw(self, raw):
        """raw: canonical host array int32[4][Nt][Ns][Ns][Ns] of binary angles (exact state)."""
        a = np.ascontiguousarray(raw, dtype=np.int32).reshape(-1)
        assert a.size == 4 * self.V
        self._ck(lib().ul_set_links_raw(self._h, _ptr(a)))

    def get_links_raw(self):
        a = np.empty((4, self.Nt, self.Ns, self.Ns, self.Ns), dtype=np.int32)
        self._ck(lib().ul_get_links_raw(self._h, _ptr(a)))
        return a

    def get_counter(self):
        v = C.c_uint64()
        self._ck(lib().ul_get_counter(self._h, C.byref(v)))
        return v.value

    def set_counter(self, v):
        self._ck(lib().ul_set_counter(self._h, int(v)))

    def sweep(self, n_hb, n_or):
        self._ck(lib().ul_sweep(self._h, int(n_hb), int(n_or)))

    def substep(self, kind, parity, mu, slab_d=0):
        self._ck(lib().ul_substep(self._h, int(kind), int(parity), int(mu), int(slab_d)))

    def substep_slabs(self, kind, parity, mu, slab_d, s_begin, s_end):
        self._ck(lib().ul_substep_slabs(self._h, int(kind), int(parity), int(mu), int(slab_d), int(s_begin), int(s_end)))

    def set_slab_group(self, n_slabs):
        self._ck(lib().ul_set_slab_group(self._h, int(n_slabs)))

    def set_slab_group_streams(self, n_streams):
        self._ck(lib().ul_set_slab_group_streams(self._h, int(n_streams)))

    def set_update_algorithm(self, alg, delta=np.pi):
        self._ck(lib().ul_set_update_algorithm(self._h, int(alg), float(delta)))

    def set_subupdate(self, n_hb, n_or, k_sweeps=1):
        self._ck(lib().ul_set_subupdate(self._h, int(n_hb), int(n_or), int(k_sweeps)))

    def set_multihit(self, on):
        self._ck(lib().ul_set_multihit(self._h, int(on)))

    def set_accum_batch(self, depth):
        self._ck(lib().ul_set_accum_batch(self._h, int(depth)))

    def multilevel(self, slab_thickness, n_sub, r_max, field_points=None):
        fp, n = _fps(field_points)
        self._ck(lib().ul_multilevel(self._h, int(slab_thickness), int(n_sub), int(r_max), _ptr(fp), n))
        self._meas = (int(r_max), n, self.Nt // int(slab_thickness))

    def multilevel_replay(self, slab_thickness, n_sub, r_max, field_points=None):
        fp, n = _fps(field_points)
        self._ck(lib().ul_multilevel_replay(self._h, int(slab_thickness), int(n_sub), int(r_max), _ptr(fp), n))
        self._meas = (int(r_max), n, self.Nt // int(slab_thickness))

    def multilevel2(self, d_in, n_in, d_out, n_out, r_max, field_points=None):
        fp, n = _fps(field_points)
        self._ck(lib().ul_multilevel2(self._h, int(d_in), int(n_in), int(d_out), int(n_out), int(r_max), _ptr(fp), n))
        self._meas = (int(r_max), n, self.Nt // int(d_out))

    def multilevel2_replay(self, d_in, n_in, d_out, n_out, r_max, field_points=None):
        fp, n = _fps(field_points)
        self._ck(lib().ul_multilevel2_replay(self._h, int(d_in), int(n_in), int(d_out), int(n_out), int(r_max), _ptr(fp), n))
        self._meas = (int(r_max), n, self.Nt // int(d_out))

    def measure_begin(self, slab_thickness, r_max, field_points=None):
        fp, n = _fps(field_points)
        self._ck(lib().ul_measure_begin(self._h, int(slab_thickness), int(r_max), _ptr(fp), n))
        self._meas = (int(r_max), n, self.Nt // int(slab_thickness))

    def accumulate(self):
        self._ck(lib().ul_accumulate(self._h))

    def measure_end(self):
        self._ck(lib().ul_measure_end(self._h))

    def measure2_begin(self, d_in, d_out, r_max, field_points=None):
        fp, n = _fps(field_points)
        self._ck(lib().ul_measure2_begin(self._h, int(d_in), int(d_out), int(r_max), _ptr(fp), n))
        self._meas = (int(r_max), n, self.Nt // int(d_out))

    def combine(self):
        self._ck(lib().ul_combine(self._h))

    def measure2_end(self):
        self._ck(lib().ul_measure2_end(self._h))

    def plaquette(self):
        out = np.zeros(3)
        self._ck(lib().ul_plaquette(self._h, _ptr(out)))
        return out

    def plaquette_noalloc(self, out):
        """out: caller's float64 CUDA tensor of 3 elements; written asynchronously on the lattice's stream (ul_plaquette_noalloc)."""
        if not out.is_cuda or out.dtype != self._torch.float64 or out.numel() < 3 or not out.is_contiguous():
            raise ValueError("out must be a contiguous float64 CUDA tensor with 3 elements")
        self._ck(lib().ul_plaquette_noalloc(self._h, C.c_void_p(out.data_ptr())))
        return out

    def read_correlators(self):
        if self._meas is None:
            self._ck(lib().ul_read_correlators(self._h, None, None, None))
        R, F, _ = self._meas
        corr = np.zeros((R, 2))
        field = np.zeros((R, max(F, 1), 12, 2))
        vac = np.zeros(12)
        self._ck(lib().ul_read_correlators(self._h, _ptr(corr), _ptr(field) if F else None, _ptr(vac)))
        return corr[:, 0] + 1j * corr[:, 1], (field[..., 0] + 1j * field[..., 1])[:, :F], vac

    def read_slab_averages(self):
        R, _, S = self._meas
        out = np.zeros((3, R, S, self.Ns ** 3, 2))
        self._ck(lib().ul_read_slab_averages(self._h, _ptr(out)))
        return out[..., 0] + 1j * out[..., 1]

    def polyakov(self, multihit=0):
        out = np.zeros(2)
        self._ck(lib().ul_polyakov(self._h, int(multihit), _ptr(out)))
        return complex(out[0], out[1])

    def set_site_offset(self, offset):
        self._ck(lib().ul_set_site_offset(self._h, int(offset)))

    def slab_partial_product(self, s_begin, s_end):
        """prod_{s_begin <= s < s_end} [T](x,s) of the last measurement: complex128 device tensor [3][r_max][Ns^3]."""
        torch = self._torch
        R = self._meas[0]
        out = torch.empty((3, R, self.Ns ** 3), dtype=torch.complex128, device=self.device)
        self._ck(lib().ul_slab_partial_product(self._h, int(s_begin), int(s_end), C.c_void_p(out.data_ptr())))
        self.sync()
        return out

    def combine_partial_products(self, parts):
        """parts: the shards' partial products in rank order (complex128 device tensors [3][r_max][Ns^3] on this GPU).
        Returns the global C(r) (complex numpy array): ordered product and lattice sum run in the library."""
        R = self._meas[0]
        parts = [p.contiguous() for p in parts]
        for p in parts:
            if not p.is_cuda or p.dtype != self._torch.complex128 or p.numel() != 3 * R * self.Ns ** 3:
                raise ValueError("partial products must be complex128 [3][r_max][Ns^3] tensors on the lattice's device")
        ptrs = (C.c_void_p * len(parts))(*[p.data_ptr() for p in parts])
        corr = np.empty((R, 2), dtype=np.float64)
        self._ck(lib().ul_combine_partial_products(self._h, ptrs, len(parts), _ptr(corr)))
        return corr[:, 0] + 1j * corr[:, 1]

    def set_halo_peers(self, dn_links_ptr, up_links_ptr, ghost_layers):
        """Device pointers (ints) to the link arrays of the shards below / above; (0, 0) switches the mode off."""
        self._ck(lib().ul_set_halo_peers(self._h, C.c_void_p(dn_links_ptr or None), C.c_void_p(up_links_ptr or None), int(ghost_layers)))

    def halo_flags(self):
        """Device pointer (int) of this context's two flag words (zeroed)."""
        p = C.c_void_p()
        self._ck(lib().ul_halo_flags(self._h, C.byref(p)))
        return p.value

    def set_halo_peer_flags(self, dn_flags_ptr, up_flags_ptr):
        self._ck(lib().ul_set_halo_peer_flags(self._h, C.c_void_p(dn_flags_ptr or None), C.c_void_p(up_flags_ptr or None)))

    def ipc_export(self):
        """(links handle bytes, offset, flags handle bytes, offset) for the neighbours' processes (after halo_flags())."""
        hl, hf = C.create_string_buffer(64), C.create_string_buffer(64)
        ol, of = C.c_uint64(), C.c_uint64()
        self._ck(lib().ul_ipc_export(self._h, hl, C.byref(ol), hf, C.byref(of)))
        return bytes(hl.raw), ol.value, bytes(hf.raw), of.value

    def ipc_open(self, handle, offset):
        """Device pointer (int) of a neighbour process's allocation + offset."""
        p = C.c_void_p()
        self._ck(lib().ul_ipc_open(self._h, C.c_char_p(handle), int(offset), C.byref(p)))
        return p.value

    def launch_count(self):
        v = C.c_uint64()
        self._ck(lib().ul_get_launch_count(self._h, C.byref(v)))
        return v.value

    def sync(self):
        self._ck(lib().ul_sync(self._h))
