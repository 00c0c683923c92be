"""Test-only helpers.  Nothing here is imported by the product or by oracle/.

Independent restatements used to PIN the oracle (they are textbook forms, written differently from the
oracle's per-pair 2x2 real rotation): complex-exponential RoPE, list-slicing splice, golden-file parser.
"""
from __future__ import annotations

import os

import numpy as np
import torch

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def golden(name: str) -> dict:
    """Parse ``key = value  # citation`` files under tests/golden/ (values are the paper's, cited per line)."""
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, v = (x.strip() for x in line.split("=", 1))
            parts = v.split()
            vals = [float(p) if any(c in p for c in ".e") else int(p) for p in parts]
            out[k] = vals[0] if len(vals) == 1 else vals
    return out


# ----------------------------------------------------------------------------- textbook RoPE (complex form)

def rope_complex(x: np.ndarray, pos, inv_freq: np.ndarray, pairing: int = 0) -> np.ndarray:
    """Textbook RoPE (Su et al.): view each pair as a complex number and multiply by exp(i * pos * theta).
    x: [..., d] float64; pos: scalar or [...] ; NeoX pairs (i, i+d/2), interleaved pairs (2i, 2i+1)."""
    x = np.asarray(x, np.float64)
    d = x.shape[-1]
    H = d // 2
    th = np.asarray(inv_freq, np.float32).astype(np.float64)
    if pairing == 0:
        z = x[..., :H] + 1j * x[..., H:]
    else:
        z = x[..., 0::2] + 1j * x[..., 1::2]
    ang = np.asarray(pos, np.float64)[..., None] * th
    z = z * np.exp(1j * ang)
    out = np.empty_like(x)
    if pairing == 0:
        out[..., :H], out[..., H:] = z.real, z.imag
    else:
        out[..., 0::2], out[..., 1::2] = z.real, z.imag
    return out


# ----------------------------------------------------------------------------- storage helpers (torch = library pin)

def to_storage(x: np.ndarray, dtype: int, scale: float = 1.0) -> np.ndarray:
    """float64 [n, W] -> uint8 [n, W*E] in the cache's storage type, through torch's converters."""
    x = np.ascontiguousarray(x, np.float64)
    if dtype == 2:
        return x.view(np.uint8).reshape(x.shape[0], -1).copy()
    t = torch.from_numpy(x)
    if dtype == 0:
        return t.to(torch.float32).to(torch.bfloat16).view(torch.uint8).numpy().reshape(x.shape[0], -1).copy()
    q = (t / scale).to(torch.float32).clamp(-448, 448).to(torch.float8_e4m3fn)
    return q.view(torch.uint8).numpy().reshape(x.shape[0], -1).copy()


def from_storage(b: np.ndarray, dtype: int, scale: float = 1.0) -> np.ndarray:
    """uint8 [n, W*E] -> float64 [n, W] through torch's converters."""
    b = np.ascontiguousarray(b, np.uint8)
    if dtype == 2:
        return b.view(np.float64).copy()
    t = torch.from_numpy(b)
    if dtype == 0:
        return t.view(torch.bfloat16).to(torch.float64).numpy()
    return t.view(torch.float8_e4m3fn).to(torch.float64).numpy() * scale


def list_splice(L_old: int, dirs):
    """Literal list-slicing definition of the edited sequence: tokens are ('o', old_index) or ('r', repl_row).
    dirs: (start, end, repl_len, repl_row) sorted, non-overlapping, ORIGINAL coordinates.  Applied right to left
    so that earlier indices stay valid -- the plain Python idiom, no running shift anywhere."""
    seq = [("o", i) for i in range(L_old)]
    for (s, e, n, row) in reversed(list(dirs)):
        seq[s:e] = [("r", row + q) for q in range(n)]
    return seq
