"""Weight-blob generator and (de)serialiser — layout only, no model arithmetic.

Blob layout (little-endian), SURVEY.md §8(b) "Weight blob":

  header, 48 bytes:
     char[4] magic "PNN1" | u32 version=1 | u32 n_species | u32 F | u32 K | u32 T
     | u32 R (readout hidden = F/2) | u32 reserved=0 | f64 rc | f64 eps_norm
  then fp64 arrays, row-major [out x in] (y = W x + b), in this order:
     Emb[n_species x F]
     for t = 1..T:  Wm1[F x F] bm1[F] Wm2[3F x F] bm2[3F] Wf[3F x K] bf[3F]
                    U[F x F] V[F x F] Wu1[F x 2F] bu1[F] Wu2[3F x F] bu2[3F]
     Wr1[R x F] br1[R] wr2[R] br2[1]
  chunk order of the 3F outputs: message/filter = [s | vs | vv]; update gate = [vv | sv | ss].

Initialisation (reading A11 in DESIGN.md): W ~ N(0, 1/fan_in), b ~ N(0, 0.1^2), Emb ~ N(0, 1);
draw order = blob order, one numpy Generator(PCG64(seed)).
"""
from __future__ import annotations

import struct
from collections import OrderedDict

import numpy as np

BLOB_MAGIC = b"PNN1"
HEADER_BYTES = 48


def blob_layout(n_species: int, F: int, K: int, T: int, R: int | None = None):
    """Ordered list of (name, shape, kind) with kind in {'emb','W','b'}; fan_in = shape[-1] for 'W'."""
    R = F // 2 if R is None else R
    out = [("Emb", (n_species, F), "emb")]
    for t in range(T):
        p = f"L{t}."
        out += [
            (p + "Wm1", (F, F), "W"), (p + "bm1", (F,), "b"),
            (p + "Wm2", (3 * F, F), "W"), (p + "bm2", (3 * F,), "b"),
            (p + "Wf", (3 * F, K), "W"), (p + "bf", (3 * F,), "b"),
            (p + "U", (F, F), "W"), (p + "V", (F, F), "W"),
            (p + "Wu1", (F, 2 * F), "W"), (p + "bu1", (F,), "b"),
            (p + "Wu2", (3 * F, F), "W"), (p + "bu2", (3 * F,), "b"),
        ]
    out += [("Wr1", (R, F), "W"), ("br1", (R,), "b"), ("wr2", (R,), "W"), ("br2", (1,), "b")]
    return out


def make_weights(n_species: int, F: int, K: int, T: int, rc: float = 5.0, eps: float = 1e-8,
                 seed: int = 0, overrides: dict | None = None) -> bytes:
    """Return the weight blob as bytes.  `overrides` maps array name -> ndarray (used by closed-form tests)."""
    R = F // 2
    rng = np.random.Generator(np.random.PCG64(seed))
    chunks = [BLOB_MAGIC, struct.pack("<7I", 1, n_species, F, K, T, R, 0), struct.pack("<2d", rc, eps)]
    for name, shape, kind in blob_layout(n_species, F, K, T, R):
        if kind == "emb":
            a = rng.standard_normal(shape)
        elif kind == "W":
            a = rng.standard_normal(shape) / np.sqrt(shape[-1])
        else:
            a = 0.1 * rng.standard_normal(shape)
        if overrides and name in overrides:
            a = np.asarray(overrides[name], dtype=np.float64).reshape(shape)
        chunks.append(np.ascontiguousarray(a, dtype="<f8").tobytes())
    return b"".join(chunks)


def parse_blob(blob: bytes):
    """Split a blob into (header dict, OrderedDict name -> fp64 ndarray).  Pure layout."""
    if blob[:4] != BLOB_MAGIC:
        raise ValueError("bad magic")
    version, n_species, F, K, T, R, _ = struct.unpack_from("<7I", blob, 4)
    rc, eps = struct.unpack_from("<2d", blob, 32)
    hdr = dict(version=version, n_species=n_species, F=F, K=K, T=T, R=R, rc=rc, eps=eps)
    arrs = OrderedDict()
    off = HEADER_BYTES
    for name, shape, _ in blob_layout(n_species, F, K, T, R):
        n = int(np.prod(shape))
        arrs[name] = np.frombuffer(blob, dtype="<f8", count=n, offset=off).reshape(shape).copy()
        off += 8 * n
    if off != len(blob):
        raise ValueError(f"blob size mismatch: parsed {off}, have {len(blob)}")
    return hdr, arrs
