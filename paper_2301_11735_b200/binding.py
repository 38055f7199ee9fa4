"""ctypes binding of libic_b200.so -- same names as include/ic.h, argument marshalling only.

PyTorch is used for device memory (the workspace tensor, trace buffers) and the CUDA stream; every step of the
path runs in the library's kernels.  There is no CPU fallback: if the library cannot be built or loaded, importing
this module raises.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

IC_OK, IC_ERR_NULL, IC_ERR_SIZE, IC_ERR_PARAM, IC_ERR_WORKSPACE, IC_ERR_CHARGE, IC_ERR_CUDA = 0, -1, -2, -3, -4, -5, -6
IC_ERR_STATIC_MAX = -7
IC_N_CLASSES = 3267
IC_STATIC_CLUSTER_MAX_L = 1024


class ic_obs(C.Structure):
    _fields_ = [("nmeas", C.c_int64), ("n2", C.c_int64), ("bV", C.c_int64), ("bJ", C.c_int64), ("M", C.c_int64),
                ("Ms", C.c_int64), ("Q", C.c_int64),
                ("sumE", C.c_double), ("sumE2", C.c_double), ("sumM", C.c_double), ("sumM2", C.c_double),
                ("sumAbsM", C.c_double), ("sumMs", C.c_double), ("sumMs2", C.c_double), ("sumAbsMs", C.c_double),
                ("T", C.c_double), ("C", C.c_double), ("chi_u", C.c_double), ("chi_s", C.c_double)]


EXPORTS = {
    "ic_workspace_bytes": (C.c_size_t, [C.c_int, C.c_int, C.c_int]),
    "ic_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_uint64,
                            C.c_int, C.c_int, C.c_void_p, C.c_size_t, C.c_void_p]),
    "ic_init_charges": (C.c_int, [C.c_void_p, C.c_int, C.c_int64, C.c_int64]),
    "ic_set_state": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "ic_sweep": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.c_int64]),
    "ic_sweep_trace": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.c_int64, C.c_void_p]),
    "ic_reset_observables": (C.c_int, [C.c_void_p]),
    "ic_observables": (C.c_int, [C.c_void_p, C.POINTER(ic_obs)]),
    "ic_state": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "ic_set_state_packed": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "ic_state_packed": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "ic_restore": (C.c_int, [C.c_void_p, C.c_int64, C.POINTER(ic_obs)]),
    "ic_debug_recompute": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_int64)]),
    "ic_thresholds": (C.c_int, [C.c_void_p, C.c_double, C.POINTER(C.c_uint32)]),
    "ic_schedule": (C.c_int, [C.c_void_p, C.c_uint64, C.POINTER(C.c_int32)]),
    "ic_maps_scratch_bytes": (C.c_size_t, [C.c_int, C.c_int64]),
    "ic_sweep_maps": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.c_int64, C.c_int64, C.c_void_p, C.c_size_t, C.c_void_p]),
    "ic_cluster_scratch_bytes": (C.c_size_t, [C.c_int]),
    "ic_largest_cluster": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_size_t, C.POINTER(C.c_int64)]),
    "ic_snapshot_ppm": (C.c_int, [C.c_void_p, C.c_int, C.c_char_p]),
    "ic_largest_cluster_static": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]),
    "ic_sweep_count": (C.c_int64, [C.c_void_p]),
    "ic_charge": (C.c_int64, [C.c_void_p]),
    "ic_set_variant": (C.c_int, [C.c_void_p, C.c_int]),
    "ic_set_max_blocks": (C.c_int, [C.c_void_p, C.c_int]),
    "ic_launch_count": (C.c_int64, [C.c_void_p]),
    "ic_kernel_family": (C.c_int, [C.c_void_p]),
    "ic_destroy": (C.c_int, [C.c_void_p]),
    "ic_strerror": (C.c_char_p, [C.c_int]),
}


def _load():
    path = _build.build()          # raises if nvcc fails; never falls back to anything else
    lib = C.CDLL(path)
    for name, (res, args) in EXPORTS.items():
        fn = getattr(lib, name)    # AttributeError if the library does not export it
        fn.restype, fn.argtypes = res, args
    return lib, path


lib, LIB_PATH = _load()


class IcError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: {lib.ic_strerror(code).decode()} (code {code})")


def _check(code, where):
    if code != IC_OK:
        raise IcError(code, where)


def largest_cluster_static(d_codes, which, d_out2, stream=None):
    """ic_largest_cluster_static: (largest cluster, number of clusters) of one lattice, without a Sim, a workspace or scratch.

    For code that cannot allocate device memory when it wants the answer (a hook inside a program that gave all of HBM to its
    own pool, a host that forbids cudaMalloc / cudaFree because they stall the device, a fixed memory budget): the scratch
    is an 8 MiB array built into the library, one per GPU, shared by all calls, so L <= IC_STATIC_CLUSTER_MAX_L (1024) and
    calls that overlap on the GPU race.  Nothing is allocated here either: the caller passes both tensors.

    d_codes: CUDA int8 tensor [L, L] of public site codes; d_out2: CUDA int64 tensor of 2 elements on the same device, written
    asynchronously on `stream` (default: torch's current stream of that device); read it after the stream has caught up.
    """
    import torch
    assert d_codes.is_cuda and d_codes.is_contiguous() and d_codes.element_size() == 1 and d_codes.dim() == 2
    assert d_out2.is_cuda and d_out2.dtype == torch.int64 and d_out2.numel() == 2 and d_out2.is_contiguous()
    assert d_out2.device == d_codes.device and d_codes.shape[0] == d_codes.shape[1]
    with torch.cuda.device(d_codes.device):              # the entry point works on the current device
        st = torch.cuda.current_stream() if stream is None else stream
        _check(lib.ic_largest_cluster_static(C.c_void_p(d_codes.data_ptr()), int(d_codes.shape[0]), int(which),
                                             C.c_void_p(d_out2.data_ptr()), C.c_void_p(st.cuda_stream)), "ic_largest_cluster_static")
    return d_out2


class Sim:
    """`replicas` copies of an L x L lattice on the current CUDA device; thin wrapper over the ic_* calls."""

    def __init__(self, L, n, delta, V, J, seed, replicas=1, bits_per_site=8, device=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2301_11735_b200 needs a CUDA device (there is no CPU path)")
        self.torch = torch
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.L, self.N, self.replicas, self.bits = int(L), int(L) * int(L), int(replicas), int(bits_per_site)
        nbytes = lib.ic_workspace_bytes(self.L, self.replicas, self.bits)
        if nbytes == 0:
            raise IcError(IC_ERR_SIZE, "ic_workspace_bytes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            aligned = (base + 255) & ~255
            self.stream = torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            _check(lib.ic_create(C.byref(h), self.L, float(n), float(delta), float(V), float(J), int(seed), self.replicas,
                                 self.bits, C.c_void_p(aligned), nbytes, C.c_void_p(self.stream.cuda_stream)), "ic_create")
        self.h = h
        self.workspace_bytes = nbytes

    # -- the boundary, one method per entry point -------------------------------------------------------------
    def init_charges(self, replica, nplus, nminus):
        _check(lib.ic_init_charges(self.h, int(replica), int(nplus), int(nminus)), "ic_init_charges")

    def set_state(self, replica, codes):
        """codes: numpy int8 [L, L] (or a pinned torch CPU tensor) of public site codes."""
        if hasattr(codes, "data_ptr"):
            assert codes.device.type == "cpu" and codes.is_contiguous() and codes.numel() == self.N and codes.element_size() == 1
            ptr = codes.data_ptr()
        else:
            codes = np.ascontiguousarray(codes, dtype=np.int8)
            assert codes.size == self.N
            ptr = codes.ctypes.data
        _check(lib.ic_set_state(self.h, int(replica), C.c_void_p(ptr)), "ic_set_state")

    def _T(self, T):
        arr = np.ascontiguousarray(np.broadcast_to(np.asarray(T, dtype=np.float64), (self.replicas,)))
        return arr, arr.ctypes.data_as(C.POINTER(C.c_double))

    def sweep(self, T, nsweeps):
        arr, p = self._T(T)
        _check(lib.ic_sweep(self.h, p, int(nsweeps)), "ic_sweep")

    def sweep_trace(self, T, nsweeps):
        """Returns a device int64 tensor [nsweeps, replicas, 6] = (n2, bV, bJ, M, Ms, Q) after every sweep."""
        arr, p = self._T(T)
        with self.torch.cuda.device(self.device), self.torch.cuda.stream(self.stream):      # the stream ic_create was given
            tr = self.torch.empty((int(nsweeps), self.replicas, 6), dtype=self.torch.int64, device=self.device)
        _check(lib.ic_sweep_trace(self.h, p, int(nsweeps), C.c_void_p(tr.data_ptr())), "ic_sweep_trace")
        return tr

    def _scratch(self, nbytes):
        """A 256-byte aligned device buffer of at least nbytes (kept and reused)."""
        if nbytes == 0:
            raise IcError(IC_ERR_SIZE, "scratch size")
        buf = getattr(self, "_scratch_buf", None)
        if buf is None or buf.numel() < nbytes + 256:
            # allocated on the context's stream: the block the old buffer gives back may still be in use by kernels queued there,
            # and the caching allocator only hands it out again to that same stream
            with self.torch.cuda.device(self.device), self.torch.cuda.stream(self.stream):
                self._scratch_buf = buf = self.torch.empty(nbytes + 256, dtype=self.torch.uint8, device=self.device)
        return (buf.data_ptr() + 255) & ~255

    def sweep_maps(self, T, nmaps, K, trace=False):
        """nmaps device-built maps of K candidate pairs each; returns the per-map trace if asked."""
        arr, p = self._T(T)
        nbytes = lib.ic_maps_scratch_bytes(self.L, int(K))
        ptr = self._scratch(nbytes)
        tr = None
        if trace:
            with self.torch.cuda.device(self.device), self.torch.cuda.stream(self.stream):
                tr = self.torch.empty((int(nmaps), self.replicas, 6), dtype=self.torch.int64, device=self.device)
        _check(lib.ic_sweep_maps(self.h, p, int(nmaps), int(K), C.c_void_p(ptr), nbytes,
                                 C.c_void_p(tr.data_ptr()) if trace else None), "ic_sweep_maps")
        return tr

    def largest_cluster(self, replica=0, which=0):
        """(size of the largest connected cluster of charged sites, number of clusters)."""
        nbytes = lib.ic_cluster_scratch_bytes(self.L)
        ptr = self._scratch(nbytes)
        out = (C.c_int64 * 2)()
        _check(lib.ic_largest_cluster(self.h, int(replica), int(which), C.c_void_p(ptr), nbytes, out), "ic_largest_cluster")
        return int(out[0]), int(out[1])

    def snapshot_ppm(self, replica, path):
        _check(lib.ic_snapshot_ppm(self.h, int(replica), os.fsencode(path)), "ic_snapshot_ppm")

    def reset_observables(self):
        _check(lib.ic_reset_observables(self.h), "ic_reset_observables")

    def observables(self):
        out = (ic_obs * self.replicas)()
        _check(lib.ic_observables(self.h, out), "ic_observables")
        return [{f: getattr(o, f) for f, _ in ic_obs._fields_} for o in out]

    def set_state_packed(self, replica, words):
        """words: numpy uint32 [L*L/16] (or a pinned torch CPU tensor of that many bytes x 4): 16 public codes per word."""
        if hasattr(words, "data_ptr"):
            assert words.device.type == "cpu" and words.is_contiguous() and words.numel() * words.element_size() == self.N // 4
            ptr = words.data_ptr()
        else:
            words = np.ascontiguousarray(words, dtype=np.uint32)
            assert words.size == self.N // 16
            ptr = words.ctypes.data
        _check(lib.ic_set_state_packed(self.h, int(replica), C.c_void_p(ptr)), "ic_set_state_packed")

    def state_packed(self, replica=0, out=None):
        if out is None:
            out = np.empty(self.N // 16, dtype=np.uint32)
        ptr = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        _check(lib.ic_state_packed(self.h, int(replica), C.c_void_p(ptr)), "ic_state_packed")
        return out

    def restore(self, sweep_count, observables):
        """ic_restore: continue a saved run -- `observables` is what observables() returned when the run was saved."""
        arr = (ic_obs * self.replicas)()
        assert len(observables) == self.replicas
        for o, d in zip(arr, observables):
            for f, _ in ic_obs._fields_:
                setattr(o, f, d[f])
        _check(lib.ic_restore(self.h, int(sweep_count), arr), "ic_restore")

    def state(self, replica=0, out=None):
        if out is None:
            out = np.empty((self.L, self.L), dtype=np.int8)
        ptr = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        _check(lib.ic_state(self.h, int(replica), C.c_void_p(ptr)), "ic_state")
        return out

    def debug_recompute(self, replica=0):
        out = (C.c_int64 * 6)()
        _check(lib.ic_debug_recompute(self.h, int(replica), out), "ic_debug_recompute")
        return np.array(list(out), dtype=np.int64)

    def thresholds(self, T):
        out = np.zeros(IC_N_CLASSES, dtype=np.uint32)
        _check(lib.ic_thresholds(self.h, float(T), out.ctypes.data_as(C.POINTER(C.c_uint32))), "ic_thresholds")
        return out

    def schedule(self, sweep):
        out = (C.c_int32 * 4)()
        _check(lib.ic_schedule(self.h, int(sweep), out), "ic_schedule")
        return tuple(out)

    def set_variant(self, variant):
        _check(lib.ic_set_variant(self.h, int(variant)), "ic_set_variant")

    def set_max_blocks(self, max_blocks):
        _check(lib.ic_set_max_blocks(self.h, int(max_blocks)), "ic_set_max_blocks")

    @property
    def sweep_count(self):
        return int(lib.ic_sweep_count(self.h))

    @property
    def Q(self):
        return int(lib.ic_charge(self.h))

    @property
    def kernel_family(self):
        """Variant number (1..6, see ic_set_variant) of the kernels the last sweep call ran; 0 before the first sweep."""
        return int(lib.ic_kernel_family(self.h))

    @property
    def launch_count(self):
        return int(lib.ic_launch_count(self.h))

    def close(self):
        if getattr(self, "h", None):
            lib.ic_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
