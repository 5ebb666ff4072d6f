"""fp64 CPU oracle for the PaiNN E/F/virial hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  The product path (paper_2506_04055_b200/) never does.  The arithmetic lives in painn_oracle.c
(plain C, fp64, brute-force neighbours, hand adjoint; see its header for the citations); this module is
argument marshalling via ctypes plus the gcc build step.  Parity with the paper at value level is
UNPINNED (no worked numbers in PAPER.md); structural pins live in tests/test_oracle_pins.py.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "painn_oracle.c")
_LIB = os.path.join(_HERE, "libpainn_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile painn_oracle.c with gcc (no FMA contraction, OpenMP).  Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_neighbors.restype = C.c_int
        _lib.oracle_compute.restype = C.c_int
        _lib.oracle_threads.restype = C.c_int
    return _lib


def threads() -> int:
    return int(_load().oracle_threads())


def _p(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def neighbors(pos, box, rc, periodic=True, smax=1):
    """Brute-force neighbour set.  Returns (i, j, image[E,3]) sorted by (i, j, image)."""
    lib = _load()
    pos = np.ascontiguousarray(pos, np.float64)
    box = np.ascontiguousarray(box, np.float64)
    N = len(pos)
    ne = C.c_longlong(0)
    lib.oracle_neighbors(_p(pos, C.c_double), C.c_longlong(N), _p(box, C.c_double), C.c_int(int(periodic)),
                         C.c_double(rc), C.c_int(smax), C.c_longlong(0), C.byref(ne), None, None, None)
    E = ne.value
    ei = np.empty(max(E, 1), np.int32); ej = np.empty(max(E, 1), np.int32); im = np.empty((max(E, 1), 3), np.int8)
    rc_ = lib.oracle_neighbors(_p(pos, C.c_double), C.c_longlong(N), _p(box, C.c_double), C.c_int(int(periodic)),
                               C.c_double(rc), C.c_int(smax), C.c_longlong(E), C.byref(ne),
                               _p(ei, C.c_int), _p(ej, C.c_int), _p(im, C.c_byte))
    if rc_ != 0:
        raise RuntimeError(f"oracle_neighbors failed: {rc_}")
    return ei[:E], ej[:E], im[:E]


def compute(blob: bytes, pos, types, box, n_local=None, n_ghost=0, ghost_owner=None, periodic=None, smax=1,
            want_states=False):
    """E, F, virial (+ per-atom energies, raw 3x3 virial, edge count, optional layer states) in fp64.

    periodic=None follows the C-ABI convention: n_ghost == 0 -> periodic box, n_ghost > 0 -> open boundaries."""
    lib = _load()
    pos = np.ascontiguousarray(pos, np.float64)
    types = np.ascontiguousarray(types, np.int32)
    box = np.ascontiguousarray(box, np.float64)
    N = len(pos)
    n_local = N - n_ghost if n_local is None else n_local
    assert n_local + n_ghost == N
    if periodic is None:
        periodic = n_ghost == 0
    go = None if ghost_owner is None else np.ascontiguousarray(ghost_owner, np.int32)
    energy = C.c_double(0.0)
    forces = np.zeros((N, 3)); virial = np.zeros(6); virial9 = np.zeros((3, 3)); ei = np.zeros(N)
    states = None
    if want_states:
        import struct
        F, K, T = struct.unpack_from("<3I", blob, 12)
        states = np.zeros((T + 1, N, 4 * F))
    ne = C.c_longlong(0)
    buf = (C.c_char * len(blob)).from_buffer_copy(blob)
    rc_ = lib.oracle_compute(buf, C.c_size_t(len(blob)), _p(pos, C.c_double), _p(types, C.c_int),
                             _p(box, C.c_double), C.c_longlong(n_local), C.c_longlong(n_ghost),
                             C.c_int(int(periodic)), C.c_int(smax), _p(go, C.c_int), C.byref(energy),
                             _p(forces, C.c_double), _p(virial, C.c_double), _p(virial9, C.c_double),
                             _p(ei, C.c_double), _p(states, C.c_double), C.byref(ne))
    if rc_ != 0:
        raise RuntimeError(f"oracle_compute failed: {rc_}")
    return dict(energy=energy.value, forces=forces, virial=virial, virial9=virial9, atom_energy=ei,
                n_edges=ne.value, states=states)
