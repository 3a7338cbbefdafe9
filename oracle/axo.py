"""ctypes binding of the CPU oracle (oracle/axo_oracle.cpp).  Test infrastructure only.

Same call names as the CUDA binding (create / place_neurons / add_source / step / read_state ...), so that the
parity tests drive both with the same code.  Holds no arithmetic of the method.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None

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


class OracleError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("axo error %d: %s" % (code, msg))
        self.code = code


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        L = _lib
        vp, u32, u64, f32 = C.c_void_p, C.c_uint32, C.c_uint64, C.c_float
        L.axo_create.argtypes = [vp, f32, u32, f32, f32, f32, u64, C.POINTER(vp)]
        L.axo_destroy.argtypes = [vp]
        L.axo_destroy.restype = None
        L.axo_last_error.argtypes = [vp]
        L.axo_last_error.restype = C.c_char_p
        L.axo_set_capacity.argtypes = [vp, u64, u32]
        L.axo_place_neurons.argtypes = [vp, vp, vp, u32]
        L.axo_add_source.argtypes = [vp, f32, f32, f32, C.c_uint8, C.c_int8, u32]
        L.axo_set_shard.argtypes = [vp, u32, u32]
        L.axo_set_steering.argtypes = [vp, C.c_int, f32, f32]
        L.axo_set_sensing.argtypes = [vp, C.c_int]
        L.axo_set_key_order.argtypes = [vp, C.c_int]
        L.axo_step.argtypes = [vp, u32]
        L.axo_step_phase.argtypes = [vp, u32]
        L.axo_load_particles.argtypes = [vp, vp, vp, vp, vp, vp, u64, u32, u32]
        L.axo_load_cones.argtypes = [vp, vp, vp, vp, vp, u32]
        L.axo_read_state.argtypes = [vp, u32, vp, C.c_size_t, C.POINTER(C.c_size_t)]
        L.axo_load_sense.argtypes = [vp, vp, vp, u32]
        L.axo_set_connect.argtypes = [vp, f32, f32]
        L.axo_load_targets.argtypes = [vp, vp, u32]
        L.axo_build_graph.argtypes = [vp, C.c_int]
        L.axo_bfs.argtypes = [vp, u32]
        L.axo_philox4x32_10.argtypes = [vp, vp, vp]
        L.axo_philox4x32_10.restype = None
        L.axo_normals.argtypes = [u64, u32, u32, u32, u32, vp, vp, vp]
        L.axo_normals.restype = None
        L.axo_sense_brute.argtypes = [vp, vp, vp]
        L.axo_bin_keys.argtypes = [vp, u32, u32, vp, vp, vp, vp]
        L.axo_stencil_S2.argtypes = [f32]
        L.axo_stencil_S2.restype = C.c_int64
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


class Oracle:
    """One oracle context; method names follow include/axg.h without the prefix."""

    def __init__(self, grid, D, emission, radius, speed, noise, seed):
        self._L = lib()
        g = (C.c_uint32 * 3)(*[int(v) for v in grid])
        h = C.c_void_p()
        rc = self._L.axo_create(g, D, emission, radius, speed, noise, seed, C.byref(h))
        if rc:
            raise OracleError(rc, self._L.axo_last_error(None).decode())
        self._h = h
        self.grid = tuple(int(v) for v in grid)

    def _chk(self, rc):
        if rc:
            raise OracleError(rc, self._L.axo_last_error(self._h).decode())

    def close(self):
        if self._h:
            self._L.axo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_capacity(self, max_particles, max_segments):
        self._chk(self._L.axo_set_capacity(self._h, int(max_particles), int(max_segments)))

    def place_neurons(self, xyz, heading=None):
        xyz = np.ascontiguousarray(xyz, dtype=np.float32).reshape(-1, 3)
        hd = None if heading is None else np.ascontiguousarray(heading, dtype=np.float32).reshape(-1, 3)
        self._chk(self._L.axo_place_neurons(self._h, _ptr(xyz), _ptr(hd), xyz.shape[0]))

    def add_source(self, x, y, z, species=0, polarity=1, rate=0):
        self._chk(self._L.axo_add_source(self._h, x, y, z, species, polarity, rate))

    def set_steering(self, mode, gain=1.0, turn=3.141592653589793 / 30):
        self._chk(self._L.axo_set_steering(self._h, int(mode), gain, turn))

    def set_key_order(self, order):
        self._chk(self._L.axo_set_key_order(self._h, int(order)))

    def set_sensing(self, mode):
        self._chk(self._L.axo_set_sensing(self._h, int(mode)))

    def set_connect(self, r_cone, r_soma):
        self._chk(self._L.axo_set_connect(self._h, r_cone, r_soma))

    def load_targets(self, target):
        target = np.ascontiguousarray(target, dtype=np.uint32)
        self._chk(self._L.axo_load_targets(self._h, _ptr(target), target.shape[0]))

    def build_graph(self, directed=False):
        self._chk(self._L.axo_build_graph(self._h, 1 if directed else 0))

    def bfs(self, root):
        self._chk(self._L.axo_bfs(self._h, int(root)))
        return self.read_state("BFS_LEVEL")

    def set_shard(self, rank, world):
        self._chk(self._L.axo_set_shard(self._h, rank, world))

    def step(self, n=1):
        self._chk(self._L.axo_step(self._h, n))

    def step_phase(self, mask):
        self._chk(self._L.axo_step_phase(self._h, mask))

    def load_particles(self, x, y, z, species, ids, next_id, step):
        x = np.ascontiguousarray(x, dtype=np.float32)
        y = np.ascontiguousarray(y, dtype=np.float32)
        z = np.ascontiguousarray(z, dtype=np.float32)
        species = np.ascontiguousarray(species, dtype=np.uint8)
        ids = np.ascontiguousarray(ids, dtype=np.uint32)
        n = x.shape[0]
        assert y.shape[0] == n and z.shape[0] == n and species.shape[0] == n and ids.shape[0] == n
        self._chk(self._L.axo_load_particles(self._h, _ptr(x), _ptr(y), _ptr(z), _ptr(species), _ptr(ids), n,
                                             int(next_id) & 0xFFFFFFFF, int(step)))

    def load_cones(self, pos, heading, state, poly_len):
        pos = np.ascontiguousarray(pos, dtype=np.float32).reshape(-1, 3)
        heading = np.ascontiguousarray(heading, dtype=np.float32).reshape(-1, 3)
        state = np.ascontiguousarray(state, dtype=np.uint8)
        poly_len = np.ascontiguousarray(poly_len, dtype=np.uint32)
        self._chk(self._L.axo_load_cones(self._h, _ptr(pos), _ptr(heading), _ptr(state), _ptr(poly_len), pos.shape[0]))

    # the sharded loop's call names (paper_1405_3331_b200/sharded.py drives either binding)
    def check_capacity(self, n):
        pass

    def enqueue_phase(self, mask):
        self.step_phase(mask)

    def sync(self):
        pass

    def load_sense(self, counts, moment):
        counts = np.ascontiguousarray(counts, dtype=np.int64)
        moment = np.ascontiguousarray(moment, dtype=np.int64)
        self._chk(self._L.axo_load_sense(self._h, _ptr(counts), _ptr(moment), counts.size // 4))

    def read_state(self, field):
        f = FIELDS[field] if isinstance(field, str) else int(field)
        n = C.c_size_t(0)
        self._chk(self._L.axo_read_state(self._h, f, None, 0, C.byref(n)))
        out = np.empty(n.value, dtype=_DTYPES[f])
        if n.value:
            self._chk(self._L.axo_read_state(self._h, f, _ptr(out), out.nbytes, C.byref(n)))
        return out

    def counters(self):
        return dict(zip(COUNTER_NAMES, (int(v) for v in self.read_state("COUNTERS"))))

    def sense_brute(self):
        nc = self.read_state("CONE_STATE").shape[0]
        counts = np.zeros((nc, 4), dtype=np.int64)
        moment = np.zeros((nc, 4, 3), dtype=np.int64)
        self._chk(self._L.axo_sense_brute(self._h, _ptr(counts), _ptr(moment)))
        return counts, moment


def philox4x32_10(ctr, key):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().axo_philox4x32_10(_ptr(ctr), _ptr(key), _ptr(out))
    return out


def normals(seed, id0, n, t, stream):
    r = np.zeros((n, 4), dtype=np.uint32)
    u = np.zeros((n, 4), dtype=np.float32)
    z = np.zeros((n, 3), dtype=np.float32)
    lib().axo_normals(int(seed), int(id0), int(n), int(t), int(stream), _ptr(r), _ptr(u), _ptr(z))
    return r, u, z


def bin_keys(keys, cells):
    keys = np.ascontiguousarray(keys, dtype=np.uint32)
    n = keys.shape[0]
    perm = np.zeros(n, dtype=np.uint32)
    ks = np.zeros(n, dtype=np.uint32)
    cs = np.zeros(cells, dtype=np.uint32)
    ce = np.zeros(cells, dtype=np.uint32)
    rc = lib().axo_bin_keys(_ptr(keys), n, cells, _ptr(perm), _ptr(ks), _ptr(cs), _ptr(ce))
    if rc:
        raise OracleError(rc, "bin_keys")
    return perm, ks, cs, ce


def stencil_S2(radius):
    return int(lib().axo_stencil_S2(radius))
