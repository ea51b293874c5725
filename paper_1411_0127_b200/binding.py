"""ctypes binding of libising_b200.so (include/ising.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch supplies device memory
(`torch.Tensor.data_ptr()`) and streams (`torch.cuda.current_stream().cuda_stream`), nothing else.
There is no CPU fallback: loading fails if the library cannot be built or found, and the device calls
raise `IsingError` on a machine without a CUDA device.
"""
from __future__ import annotations

import ctypes as C

from . import build as _build

PHILOX, MINSTD, PHILOX_SHARED = 0, 1, 2
PR_SHARED, MT19937_SHARED = 3, 4  # shared draw from stored-state lane generators (include/ising.h, R19)
LAYOUT_AUTO, LAYOUT_SAMPLE_PACKED, LAYOUT_BATCH = 0, 1, 2  # ising_create_layout
OK, EINVAL, ECUDA, ELIMIT = 0, -1, -2, -3
STATIC_MAX_L = 128  # ising_energy_static

EXPORTS = (
    "ising_workspace_bytes", "ising_create", "ising_create_layout", "ising_load_state", "ising_sweep", "ising_sweep_trace", "ising_energy",
    "ising_get_spins", "ising_run_host", "ising_run_host_async", "ising_thresholds", "ising_fnv1a64_host", "ising_fnv1a64_scratch_bytes", "ising_fnv1a64", "ising_get_t", "ising_set_t",
    "ising_set_kernel", "ising_kernel_launches", "ising_hostcheck_update_word", "ising_destroy", "ising_strerror",
    "ising_overlap", "ising_get_lanes", "ising_set_lanes", "ising_resume_lanes", "ising_prng_state_bytes", "ising_prng_init", "ising_prng_count_odd",
    "ising_slab_workspace_bytes", "ising_create_slab", "ising_slab_half_sweep_boundary", "ising_slab_half_sweep_bulk", "ising_slab_plane",
    "ising_energy_static", "ising_slab_connect", "ising_slab_half_sweep_boundary_push", "ising_slab_sweep_local_push", "ising_slab_sweep_local", "ising_sliced_scratch_bytes", "ising_sliced_begin", "ising_sliced_sweep", "ising_sliced_end",
)

_lib = None


class IsingError(RuntimeError):
    pass


def lib() -> C.CDLL:
    """Load (building first if stale) the C-ABI library and declare its prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(_build.build())
    vp, u64, i32, sz, dbl = C.c_void_p, C.c_uint64, C.c_int, C.c_size_t, C.c_double
    L.ising_workspace_bytes.argtypes = [i32, i32, i32, C.POINTER(sz)]
    L.ising_create.argtypes = [i32, i32, u64, i32, vp, sz, C.POINTER(vp)]
    L.ising_create_layout.argtypes = [i32, i32, u64, i32, i32, vp, sz, C.POINTER(vp)]
    L.ising_load_state.argtypes = [vp, vp, vp, vp]
    L.ising_sweep.argtypes = [vp, dbl, i32, vp]
    L.ising_sweep_trace.argtypes = [vp, dbl, i32, vp, vp, i32, vp]
    L.ising_energy.argtypes = [vp, vp, vp, vp]
    L.ising_get_spins.argtypes = [vp, vp, vp]
    L.ising_overlap.argtypes = [vp, i32, i32, vp, vp]
    L.ising_energy_static.argtypes = [i32, vp, vp, vp, vp, vp]
    L.ising_run_host.argtypes = [vp, vp, vp, dbl, i32, vp, vp, vp, vp]
    L.ising_run_host_async.argtypes = [vp, vp, vp, dbl, i32, vp, vp, vp, vp]
    L.ising_thresholds.argtypes = [dbl, i32, C.POINTER(u64)]
    L.ising_fnv1a64_host.argtypes = [vp, sz]
    L.ising_fnv1a64_host.restype = u64
    L.ising_fnv1a64_scratch_bytes.argtypes = [sz, C.POINTER(sz)]
    L.ising_fnv1a64.argtypes = [vp, sz, vp, sz, vp, vp]
    L.ising_get_t.argtypes = [vp, C.POINTER(u64)]
    L.ising_set_t.argtypes = [vp, u64]
    L.ising_set_kernel.argtypes = [vp, i32]
    L.ising_kernel_launches.argtypes = [vp]
    L.ising_kernel_launches.restype = u64
    L.ising_hostcheck_update_word.argtypes = [i32, u64, u64, dbl, C.POINTER(C.c_uint32), u64, u64, u64,
                                              C.POINTER(C.c_uint32)]
    L.ising_get_lanes.argtypes = [vp, C.POINTER(C.c_uint32)]
    L.ising_set_lanes.argtypes = [vp, C.c_uint32]
    L.ising_resume_lanes.argtypes = [vp, u64, C.c_uint32]
    L.ising_prng_state_bytes.argtypes = [i32, C.c_uint32, C.POINTER(sz)]
    L.ising_prng_init.argtypes = [i32, u64, C.c_uint32, vp, vp]
    L.ising_prng_count_odd.argtypes = [i32, u64, C.c_uint32, u64, u64, vp, vp, vp, vp]
    L.ising_slab_workspace_bytes.argtypes = [i32, i32, i32, C.POINTER(sz)]
    L.ising_create_slab.argtypes = [i32, i32, i32, u64, i32, vp, sz, C.POINTER(vp)]
    L.ising_slab_half_sweep_boundary.argtypes = [vp, dbl, vp]
    L.ising_slab_half_sweep_bulk.argtypes = [vp, dbl, vp]
    L.ising_slab_plane.argtypes = [vp, i32, i32, C.POINTER(vp), C.POINTER(sz)]
    L.ising_slab_sweep_local.argtypes = [C.POINTER(vp), i32, dbl, i32, vp, vp]
    L.ising_slab_sweep_local_push.argtypes = [C.POINTER(vp), i32, dbl, i32, vp, vp]
    L.ising_slab_connect.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]
    L.ising_slab_half_sweep_boundary_push.argtypes = [vp, dbl, vp]
    L.ising_sliced_scratch_bytes.argtypes = [vp, C.POINTER(sz)]
    L.ising_sliced_begin.argtypes = [vp, vp, vp]
    L.ising_sliced_sweep.argtypes = [vp, vp, dbl, i32, vp]
    L.ising_sliced_end.argtypes = [vp, vp, vp]
    L.ising_destroy.argtypes = [vp]
    L.ising_strerror.argtypes = [i32]
    L.ising_strerror.restype = C.c_char_p
    _lib = L
    return L


def _check(rc: int, what: str):
    if rc != OK:
        raise IsingError(f"{what}: {lib().ising_strerror(rc).decode()} ({rc})")


def ising_workspace_bytes(L: int, nsamples: int, rng_mode: int) -> int:
    out = C.c_size_t(0)
    _check(lib().ising_workspace_bytes(L, nsamples, rng_mode, C.byref(out)), "ising_workspace_bytes")
    return out.value


def ising_fnv1a64_scratch_bytes(nbytes: int) -> int:
    out = C.c_size_t(0)
    _check(lib().ising_fnv1a64_scratch_bytes(nbytes, C.byref(out)), "ising_fnv1a64_scratch_bytes")
    return out.value


def ising_fnv1a64(data, out=None, scratch=None, stream=None):
    """64-bit FNV-1a of the bytes of a contiguous CUDA tensor, computed on the device (include/ising.h).  Returns a one-element
    int64 CUDA tensor holding the 64 bits (asynchronous on `stream`); `out` / `scratch` may be passed to avoid allocations."""
    import torch

    assert data.is_cuda and data.is_contiguous()
    nbytes = data.numel() * data.element_size()
    need = ising_fnv1a64_scratch_bytes(nbytes)
    if scratch is None:
        scratch = torch.empty(need, dtype=torch.uint8, device=data.device)
    if out is None:
        out = torch.empty(1, dtype=torch.int64, device=data.device)
    with torch.cuda.device(data.device):
        _check(lib().ising_fnv1a64(data.data_ptr(), nbytes, scratch.data_ptr(), scratch.numel(), out.data_ptr(), _stream_ptr(stream)),
               "ising_fnv1a64")
    return out


def ising_thresholds(beta: float, rng_mode: int) -> tuple[int, int, int]:
    out = (C.c_uint64 * 3)()
    _check(lib().ising_thresholds(float(beta), rng_mode, out), "ising_thresholds")
    return tuple(int(v) for v in out)


def ising_fnv1a64_host(buf) -> int:
    """FNV-1a 64 of a contiguous numpy array / bytes object (host)."""
    import numpy as np

    a = np.ascontiguousarray(np.frombuffer(buf, dtype=np.uint8) if isinstance(buf, (bytes, bytearray)) else buf)
    return int(lib().ising_fnv1a64_host(a.ctypes.data, a.nbytes))


def ising_hostcheck_update_word(rng_mode, seed, t, beta, ops, word_index, site0=0, site_stride=2) -> int:
    arr = (C.c_uint32 * 13)(*[int(v) & 0xFFFFFFFF for v in ops])
    out = C.c_uint32(0)
    _check(lib().ising_hostcheck_update_word(rng_mode, seed, t, float(beta), arr, word_index, site0, site_stride,
                                             C.byref(out)), "ising_hostcheck_update_word")
    return out.value


def ising_prng_state_bytes(kind: int, nlanes: int) -> int:
    out = C.c_size_t(0)
    _check(lib().ising_prng_state_bytes(kind, nlanes, C.byref(out)), "ising_prng_state_bytes")
    return out.value


def ising_prng_init(kind: int, seed: int, nlanes: int, state, stream=None):
    """state: uint8 CUDA tensor of ising_prng_state_bytes bytes (None for Philox)."""
    _check(lib().ising_prng_init(kind, seed, nlanes, state.data_ptr() if state is not None else None, _stream_ptr(stream)),
           "ising_prng_init")


def ising_prng_count_odd(kind: int, seed: int, nlanes: int, ndrawn_before: int, ndraws: int, state, odd, total, stream=None):
    """odd, total: int64 CUDA tensors of nlanes elements (uint64 bit patterns)."""
    assert odd.is_cuda and total.is_cuda and odd.numel() == nlanes and total.numel() == nlanes
    _check(lib().ising_prng_count_odd(kind, seed, nlanes, ndrawn_before, ndraws, state.data_ptr() if state is not None else None,
                                      odd.data_ptr(), total.data_ptr(), _stream_ptr(stream)), "ising_prng_count_odd")


def _stream_ptr(stream=None) -> int:
    import torch

    return (stream if stream is not None else torch.cuda.current_stream()).cuda_stream


def ising_energy_static(L: int, spins, J, E, M=None, stream=None) -> None:
    """E (and M) of ONE canonical packed sample without a handle, a workspace or any allocation: the scratch is a fixed array in
    the library (include/ising.h: L a multiple of 64, L <= STATIC_MAX_L; calls that overlap on the GPU race).  spins: (L^3/32,)
    and J: (3 L^3/32,) 4-byte-element CUDA tensors; E, M: caller-owned one-element int64 CUDA tensors, written asynchronously on
    `stream` (default: torch's current stream) of the tensors' device.  Nothing is allocated here either."""
    import torch

    assert spins.is_cuda and J.is_cuda and E.is_cuda and E.dtype == torch.int64 and (M is None or (M.is_cuda and M.dtype == torch.int64))
    assert spins.is_contiguous() and J.is_contiguous() and spins.numel() * 32 == L**3 and J.numel() * 32 == 3 * L**3 or L % 64 != 0 or L > STATIC_MAX_L
    with torch.cuda.device(spins.device):
        _check(lib().ising_energy_static(int(L), spins.data_ptr(), J.data_ptr(), E.data_ptr(), M.data_ptr() if M is not None else None,
                                         _stream_ptr(stream)), "ising_energy_static")


def _u32(t):
    """View a 4-byte-element CUDA/CPU tensor's storage as a raw pointer (uint32 words)."""
    return t.data_ptr()


class Ising:
    """Handle of one simulation: `ising_create` .. `ising_destroy` with torch tensors as buffers.

    spins / couplings are torch int32 (or uint32) CUDA tensors in the canonical packed format:
    spins (nsamples, W), couplings (nsamples, 3, W), W = ceil(L^3/32).
    """

    def __init__(self, L: int, nsamples: int = 1, seed: int = 0, rng_mode: int = PHILOX, device=None, workspace=None,
                 layout: int = LAYOUT_AUTO):
        """`device`: the CUDA device of the handle (default: torch's current device, so that a process that has called
        torch.cuda.set_device(LOCAL_RANK) gets its own GPU).  `workspace`: optional caller-owned uint8 CUDA tensor of at least
        ising_workspace_bytes bytes, 256-byte aligned (default: allocated here, on `device`).  Every call of the handle runs
        with `device` current, takes its default stream from that device and rejects tensors that live elsewhere; the library
        itself refuses a handle whose workspace is not on the current device (ISING_EINVAL)."""
        import torch

        self.L, self.nsamples, self.seed, self.rng_mode, self.layout = L, nsamples, seed, rng_mode, layout
        self.N = L ** 3
        self.W = (self.N + 31) // 32
        nbytes = ising_workspace_bytes(L, nsamples, rng_mode)
        if workspace is None:
            dev = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
            if dev.index is None:
                dev = torch.device("cuda", torch.cuda.current_device())
            self.device = dev
            # torch's caching allocator returns 512-byte aligned blocks
            workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        else:
            assert workspace.is_cuda and workspace.dtype == torch.uint8 and workspace.is_contiguous()
            assert device is None or torch.device(device) == workspace.device, "workspace is not on `device`"
            self.device = workspace.device
            nbytes = workspace.numel()
        self.workspace = workspace
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            _check(lib().ising_create_layout(L, nsamples, seed, rng_mode, layout, self.workspace.data_ptr(), nbytes, C.byref(h)),
                   "ising_create_layout")
        self._h = h

    def _on_device(self, *tensors):
        """Guard for the device calls: makes the handle's device current (so that the launches, and the default stream, are
        that device's) and checks that every CUDA tensor handed in lives on it."""
        import torch

        for x in tensors:
            assert x is None or not x.is_cuda or x.device == self.device, \
                f"tensor on {x.device}, handle on {self.device}: a kernel would dereference another GPU's memory"
        return torch.cuda.device(self.device)

    # -- the C-ABI calls, same names
    def ising_load_state(self, spins, J, stream=None):
        assert spins.is_cuda and J.is_cuda and spins.is_contiguous() and J.is_contiguous()
        assert spins.numel() == self.nsamples * self.W and J.numel() == 3 * self.nsamples * self.W
        with self._on_device(spins, J):
            _check(lib().ising_load_state(self._h, _u32(spins), _u32(J), _stream_ptr(stream)), "ising_load_state")

    def ising_sweep(self, beta: float, nsweeps: int, stream=None):
        with self._on_device():
            _check(lib().ising_sweep(self._h, float(beta), int(nsweeps), _stream_ptr(stream)), "ising_sweep")

    def ising_sweep_trace(self, beta: float, nsweeps: int, every_half_sweeps: int = 1, want_M: bool = True, stream=None):
        """Returns (E, M) int64 CUDA tensors of shape (records, nsamples)."""
        import torch

        nrec = (2 * nsweeps) // every_half_sweeps
        E = torch.empty((nrec, self.nsamples), dtype=torch.int64, device=self.device)
        M = torch.empty((nrec, self.nsamples), dtype=torch.int64, device=self.device) if want_M else None
        with self._on_device():
            _check(lib().ising_sweep_trace(self._h, float(beta), int(nsweeps), E.data_ptr(), M.data_ptr() if want_M else None,
                                           int(every_half_sweeps), _stream_ptr(stream)), "ising_sweep_trace")
        return E, M

    def ising_energy(self, stream=None):
        """Returns (E, M) int64 CUDA tensors of shape (nsamples,)."""
        import torch

        E = torch.empty(self.nsamples, dtype=torch.int64, device=self.device)
        M = torch.empty(self.nsamples, dtype=torch.int64, device=self.device)
        with self._on_device():
            _check(lib().ising_energy(self._h, E.data_ptr(), M.data_ptr(), _stream_ptr(stream)), "ising_energy")
        return E, M

    def ising_overlap(self, sample_a: int, sample_b: int, stream=None):
        """Returns q_ab as a one-element int64 CUDA tensor."""
        import torch

        q = torch.empty(1, dtype=torch.int64, device=self.device)
        with self._on_device():
            _check(lib().ising_overlap(self._h, int(sample_a), int(sample_b), q.data_ptr(), _stream_ptr(stream)), "ising_overlap")
        return q

    def ising_get_spins(self, out=None, stream=None):
        import torch

        if out is None:
            out = torch.empty((self.nsamples, self.W), dtype=torch.int32, device=self.device)
        assert out.is_cuda and out.is_contiguous() and out.numel() == self.nsamples * self.W
        with self._on_device(out):
            _check(lib().ising_get_spins(self._h, _u32(out), _stream_ptr(stream)), "ising_get_spins")
        return out

    def ising_run_host(self, h_spins, h_J, beta: float, nsweeps: int, h_spins_out=None, stream=None):
        """Host tensors in (ideally pinned), host results out; returns (E, M) int64 CPU tensors."""
        import torch

        assert not h_spins.is_cuda and not h_J.is_cuda
        E = torch.empty(self.nsamples, dtype=torch.int64).pin_memory()
        M = torch.empty(self.nsamples, dtype=torch.int64).pin_memory()
        with self._on_device():
            _check(lib().ising_run_host(self._h, _u32(h_spins), _u32(h_J), float(beta), int(nsweeps),
                                        _u32(h_spins_out) if h_spins_out is not None else None, E.data_ptr(), M.data_ptr(),
                                        _stream_ptr(stream)), "ising_run_host")
        return E, M

    def ising_run_host_async(self, h_spins, h_J, beta: float, nsweeps: int, h_spins_out, h_E, h_M=None, stream=None):
        """Enqueue the ising_run_host job on `stream` and return at once.  Every tensor must be a pinned CPU tensor the caller
        keeps alive; results (h_spins_out, h_E, h_M) are valid after the stream has been synchronised."""
        for x in (h_spins, h_J, h_spins_out, h_E, h_M):
            assert x is None or (not x.is_cuda and x.is_pinned()), "ising_run_host_async needs pinned host tensors"
        with self._on_device():
            _check(lib().ising_run_host_async(self._h, _u32(h_spins), _u32(h_J), float(beta), int(nsweeps),
                                              _u32(h_spins_out) if h_spins_out is not None else None, h_E.data_ptr(),
                                              h_M.data_ptr() if h_M is not None else None, _stream_ptr(stream)),
                   "ising_run_host_async")

    # -- the paper's sliced layout beside the handle's own (include/ising.h)
    def ising_sliced_begin(self, stream=None):
        """Allocates the scratch on first use and copies the handle's state into the sliced layout."""
        import torch

        if getattr(self, "_sliced", None) is None:
            n = C.c_size_t(0)
            _check(lib().ising_sliced_scratch_bytes(self._h, C.byref(n)), "ising_sliced_scratch_bytes")
            self._sliced = torch.empty(n.value, dtype=torch.uint8, device=self.device)
        with self._on_device():
            _check(lib().ising_sliced_begin(self._h, self._sliced.data_ptr(), _stream_ptr(stream)), "ising_sliced_begin")

    def ising_sliced_sweep(self, beta: float, nsweeps: int, stream=None):
        with self._on_device():
            _check(lib().ising_sliced_sweep(self._h, self._sliced.data_ptr(), float(beta), int(nsweeps), _stream_ptr(stream)), "ising_sliced_sweep")

    def ising_sliced_end(self, stream=None):
        with self._on_device():
            _check(lib().ising_sliced_end(self._h, self._sliced.data_ptr(), _stream_ptr(stream)), "ising_sliced_end")

    def ising_get_t(self) -> int:
        t = C.c_uint64(0)
        _check(lib().ising_get_t(self._h, C.byref(t)), "ising_get_t")
        return t.value

    def ising_set_t(self, t: int):
        _check(lib().ising_set_t(self._h, int(t)), "ising_set_t")

    def ising_get_lanes(self) -> int:
        n = C.c_uint32(0)
        _check(lib().ising_get_lanes(self._h, C.byref(n)), "ising_get_lanes")
        return n.value

    def ising_set_lanes(self, nlanes: int):
        _check(lib().ising_set_lanes(self._h, int(nlanes)), "ising_set_lanes")

    def ising_resume_lanes(self, t: int, nlanes: int):
        _check(lib().ising_resume_lanes(self._h, int(t), int(nlanes)), "ising_resume_lanes")

    def ising_set_kernel(self, which: int):
        _check(lib().ising_set_kernel(self._h, int(which)), "ising_set_kernel")

    def ising_kernel_launches(self) -> int:
        return int(lib().ising_kernel_launches(self._h))

    def ising_destroy(self):
        if self._h:
            lib().ising_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.ising_destroy()
        except Exception:
            pass


def ising_slab_workspace_bytes(L: int, nslabs: int, rng_mode: int) -> int:
    out = C.c_size_t(0)
    _check(lib().ising_slab_workspace_bytes(L, nslabs, rng_mode, C.byref(out)), "ising_slab_workspace_bytes")
    return out.value


class IsingSlab(Ising):
    """Handle of one z-slab of an L^3 lattice cut into `nslabs` slabs (include/ising.h, "z-slab decomposition").
    ising_load_state / ising_get_spins take the canonical arrays of the WHOLE lattice (the slab reads / writes its own planes);
    ising_energy returns the slab's share of E and M (the shares of all slabs add up)."""

    def __init__(self, L: int, nslabs: int, slab: int, seed: int = 0, rng_mode: int = PHILOX, device=None):
        import torch

        self.L, self.nsamples, self.seed, self.rng_mode = L, 1, seed, rng_mode
        self.nslabs, self.slab = nslabs, slab
        self.N = L ** 3
        self.W = (self.N + 31) // 32
        nbytes = ising_slab_workspace_bytes(L, nslabs, rng_mode)
        dev = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        if dev.index is None:
            dev = torch.device("cuda", torch.cuda.current_device())
        self.device = dev
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            _check(lib().ising_create_slab(L, nslabs, slab, seed, rng_mode, self.workspace.data_ptr(), nbytes, C.byref(h)),
                   "ising_create_slab")
        self._h = h

    def ising_slab_half_sweep_boundary(self, beta: float, stream=None):
        with self._on_device():
            _check(lib().ising_slab_half_sweep_boundary(self._h, float(beta), _stream_ptr(stream)), "ising_slab_half_sweep_boundary")

    def ising_slab_connect(self, below, above):
        """Fused exchange: `below` / `above` are the neighbouring IsingSlab handles (same process; their workspaces must be
        addressable from this slab's device) or pairs of raw device addresses (colour 0, colour 1) of the upper halo of the slab
        below / the lower halo of the slab above (e.g. opened from CUDA IPC handles)."""
        def addresses(x, which):
            if isinstance(x, IsingSlab):
                out = []
                for c in (0, 1):
                    ptr, nbytes = C.c_void_p(), C.c_size_t(0)
                    _check(lib().ising_slab_plane(x._h, c, which, C.byref(ptr), C.byref(nbytes)), "ising_slab_plane")
                    out.append(ptr.value)
                return out
            return [int(v) for v in x]
        dn = (C.c_void_p * 2)(*addresses(below, 3))
        up = (C.c_void_p * 2)(*addresses(above, 2))
        _check(lib().ising_slab_connect(self._h, dn, up), "ising_slab_connect")

    def ising_slab_half_sweep_boundary_push(self, beta: float, stream=None):
        with self._on_device():
            _check(lib().ising_slab_half_sweep_boundary_push(self._h, float(beta), _stream_ptr(stream)), "ising_slab_half_sweep_boundary_push")

    def ising_slab_half_sweep_bulk(self, beta: float, stream=None):
        with self._on_device():
            _check(lib().ising_slab_half_sweep_bulk(self._h, float(beta), _stream_ptr(stream)), "ising_slab_half_sweep_bulk")

    def ising_slab_plane(self, colour: int, which: int):
        """The plane as a uint8 view of the workspace: which = 0 first owned plane, 1 last owned plane (to send), 2 lower halo,
        3 upper halo (to receive into)."""
        ptr, nbytes = C.c_void_p(), C.c_size_t(0)
        _check(lib().ising_slab_plane(self._h, int(colour), int(which), C.byref(ptr), C.byref(nbytes)), "ising_slab_plane")
        off = ptr.value - self.workspace.data_ptr()
        return self.workspace[off:off + nbytes.value]


def ising_slab_sweep_local(slabs, beta: float, nsweeps: int, stream_a, stream_b, push: bool = False):
    """All slabs of a lattice in this process on one device: nsweeps sweeps, boundary kernels and plane copies on stream_a, bulk
    kernels on stream_b (the paper's Fig. 10 with device-to-device copies as the exchange).  push: the exchange fused into the
    boundary kernels (they store their end planes into the neighbours' halos), no copies."""
    arr = (C.c_void_p * len(slabs))(*[s._h for s in slabs])
    fn = lib().ising_slab_sweep_local_push if push else lib().ising_slab_sweep_local
    with slabs[0]._on_device():
        _check(fn(arr, len(slabs), float(beta), int(nsweeps), stream_a.cuda_stream, stream_b.cuda_stream), "ising_slab_sweep_local")
