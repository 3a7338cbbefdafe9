"""ctypes binding of the C-ABI library include/axg.h (libaxg.so).  Argument marshalling only: every step of the
path runs in the CUDA kernels.  There is no fallback: a missing library or a missing GPU raises.

PyTorch is used for device memory (its caching allocator backs every device buffer of a context through
`axg_set_allocator`) and for the stream (`axg_set_stream` gets torch's current stream).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

FIELDS = dict(
    COUNTERS=0, PART_X=1, PART_Y=2, PART_Z=3, PART_SPECIES=4, PART_ID=5, KEYS_SORTED=6, PERM=7, CELL_START=8,
    CELL_END=9, CONE_POS=10, CONE_HEADING=11, CONE_STATE=12, CONE_COUNTS=13, CONE_MOMENT=14, CONE_GRADIENT=15,
    POLY_LEN=16, POLYLINE=17, PRE_X=18, PRE_Y=19, PRE_Z=20, PRE_SPECIES=21, PRE_ID=22, PRE_KEY=23,
    CONE_TARGET=24, GRAPH_VA=25, GRAPH_EA=26, BFS_LEVEL=27,
)
_DTYPES = {
    0: np.uint64, 1: np.float32, 2: np.float32, 3: np.float32, 4: np.uint8, 5: np.uint32, 6: np.uint32, 7: np.uint32,
    8: np.uint32, 9: np.uint32, 10: np.float32, 11: np.float32, 12: np.uint8, 13: np.int64, 14: np.int64,
    15: np.float32, 16: np.uint32, 17: np.float32, 18: np.float32, 19: np.float32, 20: np.float32, 21: np.uint8,
    22: np.uint32, 23: np.uint32, 24: np.uint32, 25: np.uint32, 26: np.uint32, 27: np.int32,
}
PHASE_DIFFUSE, PHASE_BIN, PHASE_SENSE, PHASE_ADVANCE, PHASE_COMMIT, PHASE_ALL = 1, 2, 4, 8, 16, 31
PHASE_CONNECT = 32
NO_TARGET = 0xFFFFFFFF
COUNTER_NAMES = ("step", "n_live", "next_id", "emitted", "absorbed", "active", "arrived", "exited", "connected")
KERNEL_NAMES = ("clear", "diffuse", "emit", "sort", "reorder", "sense", "advance", "commit", "scan", "place", "settle")
BIN_AUTO, BIN_RADIX, BIN_COUNT = 0, 1, 2
STEER_VECTOR, STEER_SNR = 0, 1
SENSE_CELL, SENSE_PARTICLE, SENSE_PARTICLE_WEIGHTED = 0, 1, 2
KEY_LINEAR, KEY_BRICK, KEY_MORTON = 0, 1, 2
AUTO_COUNT_MAX_CELLS = 1 << 31   # include/axg.h AXG_AUTO_COUNT_MAX_CELLS
EXPORTS = (
    "axg_create", "axg_place_neurons", "axg_add_source", "axg_step", "axg_read_state", "axg_destroy",
    "axg_last_error", "axg_set_capacity", "axg_load_particles", "axg_load_cones", "axg_step_phase", "axg_set_shard",
    "axg_sense_buffer", "axg_set_stream", "axg_set_allocator", "axg_last_step_stats", "axg_profile_next_step",
    "axg_kernel_times", "axg_check_capacity", "axg_enqueue_phase", "axg_sync", "axg_set_binning",
    "axg_set_steering",
    "axg_set_sensing",
    "axg_set_key_order",
    "axg_get_binning",
    "axg_set_connect", "axg_load_targets", "axg_build_graph", "axg_bfs",
    "axg_enqueue_phase_on", "axg_params_fingerprint",
    "axg_bfs_noalloc",
)
BFS_NOALLOC_MAX_VERTICES = 1 << 20   # include/axg.h AXG_BFS_NOALLOC_MAX_VERTICES

_ALLOC_T = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
_FREE_T = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)

_lib = None
_hooks = None  # keeps the ctypes callbacks alive


class AxgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("axg error %d: %s" % (code, msg))
        self.code = code


class _Grid(C.Structure):
    _fields_ = [("nx", C.c_uint32), ("ny", C.c_uint32), ("nz", C.c_uint32)]


def lib_path():
    return _build.LIB


def lib(build=True):
    """Load libaxg.so (building it first if it is stale and nvcc is here).  Raises if it cannot be loaded."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if build and _build.stale() and os.path.exists(_build.NVCC):
        _build.build()
    if not os.path.exists(path):
        raise ImportError("libaxg.so is not built (python -m paper_1405_3331_b200.build); there is no fallback")
    L = C.CDLL(path)
    vp, u32, u64, f32, sz = C.c_void_p, C.c_uint32, C.c_uint64, C.c_float, C.c_size_t
    L.axg_create.argtypes = [C.POINTER(_Grid), f32, u32, f32, f32, f32, u64, C.POINTER(vp)]
    L.axg_destroy.argtypes = [vp]
    L.axg_destroy.restype = None
    L.axg_last_error.argtypes = [vp]
    L.axg_last_error.restype = C.c_char_p
    L.axg_set_capacity.argtypes = [vp, u64, u32]
    L.axg_place_neurons.argtypes = [vp, vp, vp, u32]
    L.axg_add_source.argtypes = [vp, f32, f32, f32, C.c_uint8, C.c_int8, u32]
    L.axg_set_shard.argtypes = [vp, u32, u32]
    L.axg_step.argtypes = [vp, u32]
    L.axg_step_phase.argtypes = [vp, u32]
    L.axg_check_capacity.argtypes = [vp, u32]
    L.axg_enqueue_phase.argtypes = [vp, u32]
    L.axg_sync.argtypes = [vp]
    L.axg_enqueue_phase_on.argtypes = [vp, u32, vp, C.c_int]
    L.axg_params_fingerprint.argtypes = [vp, C.POINTER(u64)]
    L.axg_set_binning.argtypes = [vp, C.c_int]
    L.axg_get_binning.argtypes = [vp, C.POINTER(C.c_int)]
    L.axg_set_connect.argtypes = [vp, f32, f32]
    L.axg_load_targets.argtypes = [vp, vp, u32]
    L.axg_build_graph.argtypes = [vp, C.c_int]
    L.axg_bfs.argtypes = [vp, u32]
    L.axg_bfs_noalloc.argtypes = [vp, vp, u32, u32, vp, vp]
    L.axg_set_steering.argtypes = [vp, C.c_int, C.c_float, C.c_float]
    L.axg_set_sensing.argtypes = [vp, C.c_int]
    L.axg_set_key_order.argtypes = [vp, C.c_int]
    L.axg_load_particles.argtypes = [vp, vp, vp, vp, vp, vp, u64, u32, u32]
    L.axg_load_cones.argtypes = [vp, vp, vp, vp, vp, u32]
    L.axg_read_state.argtypes = [vp, u32, vp, sz, C.POINTER(sz)]
    L.axg_sense_buffer.argtypes = [vp, C.POINTER(vp), C.POINTER(sz)]
    L.axg_set_stream.argtypes = [vp, vp]
    L.axg_set_allocator.argtypes = [_ALLOC_T, _FREE_T, vp]
    L.axg_last_step_stats.argtypes = [vp, C.POINTER(f32), C.POINTER(u64), C.POINTER(u64)]
    L.axg_profile_next_step.argtypes = [vp, C.c_int]
    L.axg_kernel_times.argtypes = [vp, vp]
    _lib = L
    return L


def bfs_noalloc(va_ptr, ea_ptr, n_vertices, root, level_ptr, cuda_stream=0):
    """axg_bfs_noalloc: BFS over a device-resident adjacency list with the library's fixed scratch array; allocates
    nothing.  All pointers are DEVICE addresses (ints); `level_ptr` receives int32[n_vertices]."""
    L = lib()
    rc = L.axg_bfs_noalloc(int(va_ptr), int(ea_ptr), int(n_vertices), int(root), int(level_ptr), int(cuda_stream or 0))
    if rc:
        raise AxgError(rc, L.axg_last_error(None).decode())


def use_torch_allocator():
    """Route every device allocation of the library to PyTorch's CUDA caching allocator (process-wide)."""
    global _hooks
    if _hooks is not None:
        return
    import torch

    def _alloc(nbytes, stream, _user):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
        except Exception:
            return None

    def _free(ptr, _user):
        try:
            if ptr:
                torch.cuda.caching_allocator_delete(int(ptr))
        except Exception:      # interpreter shutdown: torch is already gone, the process is about to free everything
            pass

    _hooks = (_ALLOC_T(_alloc), _FREE_T(_free))
    rc = lib().axg_set_allocator(_hooks[0], _hooks[1], None)
    if rc:
        raise AxgError(rc, "axg_set_allocator")


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


class Axg:
    """One context; method names follow include/axg.h without the prefix."""

    def __init__(self, grid, D, emission, radius, speed, noise, seed, torch_memory=True):
        self._L = lib()
        self._h = None
        stream = 0
        if torch_memory:
            import torch
            if not torch.cuda.is_available():
                raise AxgError(-4, "no CUDA device: this library has no CPU fallback")
            torch.cuda.init()
            use_torch_allocator()
            stream = torch.cuda.current_stream().cuda_stream
        g = _Grid(*[int(v) for v in grid])
        h = C.c_void_p()
        rc = self._L.axg_create(C.byref(g), D, emission, radius, speed, noise, seed, C.byref(h))
        if rc:
            raise AxgError(rc, self._L.axg_last_error(None).decode())
        self._h = h
        self.grid = tuple(int(v) for v in grid)
        if stream:
            self._chk(self._L.axg_set_stream(self._h, stream))

    def _chk(self, rc):
        if rc:
            raise AxgError(rc, self._L.axg_last_error(self._h).decode())

    def close(self):
        if self._h:
            self._L.axg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_stream(self, cuda_stream):
        self._chk(self._L.axg_set_stream(self._h, int(cuda_stream)))

    def set_capacity(self, max_particles, max_segments):
        self._chk(self._L.axg_set_capacity(self._h, int(max_particles), int(max_segments)))

    def place_neurons(self, xyz, heading=None):
        xyz = np.ascontiguousarray(xyz, dtype=np.float32).reshape(-1, 3)
        hd = None if heading is None else np.ascontiguousarray(heading, dtype=np.float32).reshape(-1, 3)
        self._chk(self._L.axg_place_neurons(self._h, _ptr(xyz), _ptr(hd), xyz.shape[0]))

    def add_source(self, x, y, z, species=0, polarity=1, rate=0):
        self._chk(self._L.axg_add_source(self._h, x, y, z, species, polarity, rate))

    def set_binning(self, mode):
        self._chk(self._L.axg_set_binning(self._h, int(mode)))

    def get_binning(self):
        mode = C.c_int(0)
        self._chk(self._L.axg_get_binning(self._h, C.byref(mode)))
        return mode.value

    def set_key_order(self, order):
        self._chk(self._L.axg_set_key_order(self._h, int(order)))

    def set_sensing(self, mode):
        self._chk(self._L.axg_set_sensing(self._h, int(mode)))

    def set_steering(self, mode, gain=1.0, turn=3.141592653589793 / 30):
        self._chk(self._L.axg_set_steering(self._h, int(mode), gain, turn))

    def set_connect(self, r_cone, r_soma):
        self._chk(self._L.axg_set_connect(self._h, r_cone, r_soma))

    def load_targets(self, target):
        target = np.ascontiguousarray(target, dtype=np.uint32)
        self._chk(self._L.axg_load_targets(self._h, _ptr(target), target.shape[0]))

    def build_graph(self, directed=False):
        self._chk(self._L.axg_build_graph(self._h, 1 if directed else 0))

    def bfs(self, root):
        self._chk(self._L.axg_bfs(self._h, int(root)))
        return self.read_state("BFS_LEVEL")

    def set_shard(self, rank, world):
        self._chk(self._L.axg_set_shard(self._h, rank, world))

    def step(self, n=1):
        self._chk(self._L.axg_step(self._h, n))

    def step_phase(self, mask):
        self._chk(self._L.axg_step_phase(self._h, mask))

    def check_capacity(self, n):
        self._chk(self._L.axg_check_capacity(self._h, n))

    def enqueue_phase(self, mask):
        self._chk(self._L.axg_enqueue_phase(self._h, mask))

    def sync(self):
        self._chk(self._L.axg_sync(self._h))

    def enqueue_phase_on(self, mask, cuda_stream, overlapped=False):
        self._chk(self._L.axg_enqueue_phase_on(self._h, mask, int(cuda_stream), 1 if overlapped else 0))

    def params_fingerprint(self):
        fp = C.c_uint64(0)
        self._chk(self._L.axg_params_fingerprint(self._h, C.byref(fp)))
        return fp.value

    def load_particles(self, x, y, z, species, ids, next_id, step):
        x = np.ascontiguousarray(x, dtype=np.float32)
        y = np.ascontiguousarray(y, dtype=np.float32)
        z = np.ascontiguousarray(z, dtype=np.float32)
        species = np.ascontiguousarray(species, dtype=np.uint8)
        ids = np.ascontiguousarray(ids, dtype=np.uint32)
        n = x.shape[0]
        assert y.shape[0] == n and z.shape[0] == n and species.shape[0] == n and ids.shape[0] == n
        self._chk(self._L.axg_load_particles(self._h, _ptr(x), _ptr(y), _ptr(z), _ptr(species), _ptr(ids), n,
                                             int(next_id) & 0xFFFFFFFF, int(step)))

    def load_cones(self, pos, heading, state, poly_len):
        pos = np.ascontiguousarray(pos, dtype=np.float32).reshape(-1, 3)
        heading = np.ascontiguousarray(heading, dtype=np.float32).reshape(-1, 3)
        state = np.ascontiguousarray(state, dtype=np.uint8)
        poly_len = np.ascontiguousarray(poly_len, dtype=np.uint32)
        self._chk(self._L.axg_load_cones(self._h, _ptr(pos), _ptr(heading), _ptr(state), _ptr(poly_len), pos.shape[0]))

    def read_state(self, field, out=None):
        f = FIELDS[field] if isinstance(field, str) else int(field)
        n = C.c_size_t(0)
        self._chk(self._L.axg_read_state(self._h, f, None, 0, C.byref(n)))
        if out is None:
            out = np.empty(n.value, dtype=_DTYPES[f])
        assert out.dtype == _DTYPES[f] and out.size >= n.value
        if n.value:
            self._chk(self._L.axg_read_state(self._h, f, _ptr(out), out.nbytes, C.byref(n)))
        return out[: n.value]

    def counters(self):
        return dict(zip(COUNTER_NAMES, (int(v) for v in self.read_state("COUNTERS"))))

    def sense_buffer(self):
        p, b = C.c_void_p(), C.c_size_t()
        self._chk(self._L.axg_sense_buffer(self._h, C.byref(p), C.byref(b)))
        return p.value, b.value

    def last_step_stats(self):
        ms, ln, ps = C.c_float(), C.c_uint64(), C.c_uint64()
        self._chk(self._L.axg_last_step_stats(self._h, C.byref(ms), C.byref(ln), C.byref(ps)))
        return dict(device_ms=ms.value, launches=ln.value, particle_steps=ps.value)

    def profile_next_step(self, enable=True):
        self._chk(self._L.axg_profile_next_step(self._h, 1 if enable else 0))

    def kernel_times(self):
        t = np.zeros(len(KERNEL_NAMES), dtype=np.float32)
        self._chk(self._L.axg_kernel_times(self._h, _ptr(t)))
        return dict(zip(KERNEL_NAMES, (float(v) for v in t)))
