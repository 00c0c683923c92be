"""Seeded synthetic inputs shared by the tests, bench.py and smoke() -- and by nothing else.

This module holds NONE of the method's arithmetic: no Delta rule, no segment logic, no rotation, no codec.
It only produces the *inputs* both the CUDA library and the CPU oracle consume: cache shapes, page tables,
free lists, directive lists, the theta table (``inv_freq``; reading G9: theta_i IS the caller's
fp32 table) and random cache / replacement bytes.  It imports neither ``oracle`` nor the binding.

The paper's workloads need SGLang, model weights and debug-gym traces; none
exist here, so these inputs stand in for them, shaped like DeepSeek-V2-Lite / V3 MLA pools
((512 + 64) x n_layers x 2 B per token) with the edit shapes of BASELINE.json's five
configs and of the paper's randomised edit suites.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

AMORTIZE, FORGET = 0, 1
DT_BF16, DT_FP8 = 0, 1
NEOX, INTERLEAVED = 0, 1


# ----------------------------------------------------------------------------- theta tables (inputs)

def rope_inv_freq(rope_dim: int = 64, base: float = 10000.0) -> np.ndarray:
    """theta_i = base^(-2i/d), i in [0, d/2), built in fp64 and rounded once to fp32 (BASELINE.json config 1)."""
    i = np.arange(rope_dim // 2, dtype=np.float64)
    return (base ** (-2.0 * i / rope_dim)).astype(np.float32)


def yarn_inv_freq(rope_dim: int = 64, base: float = 10000.0, factor: float = 40.0, orig_ctx: int = 4096,
                  beta_fast: float = 32.0, beta_slow: float = 1.0) -> np.ndarray:
    """YaRN NTK-by-parts frequencies (BASELINE.json config 3; reading G9).  Built in fp64, rounded to
    fp32.  f_e = base^(-2i/d); f_i = f_e / factor; dim(n) = d ln(orig/(2 pi n)) / (2 ln base);
    low = max(floor(dim(beta_fast)),0); high = min(ceil(dim(beta_slow)), d-1);
    ramp_i = clamp((i-low)/(high-low),0,1); theta_i = f_i ramp_i + f_e (1-ramp_i).  No mscale (G10)."""
    d = rope_dim
    i = np.arange(d // 2, dtype=np.float64)
    f_e = base ** (-2.0 * i / d)
    f_i = f_e / factor

    def dim_of(n):
        return d * math.log(orig_ctx / (2.0 * math.pi * n)) / (2.0 * math.log(base))

    low = max(math.floor(dim_of(beta_fast)), 0)
    high = min(math.ceil(dim_of(beta_slow)), d - 1)
    if high == low:
        high = low + 0.001
    ramp = np.clip((i - low) / (high - low), 0.0, 1.0)
    return (f_i * ramp + f_e * (1.0 - ramp)).astype(np.float32)


# ----------------------------------------------------------------------------- workload description

@dataclass
class Workload:
    name: str
    n_layers: int
    seq_lens: list                      # per request
    page_size: int
    dtype: int = DT_BF16
    pairing: int = NEOX
    layer_pairing: list = None          # per-layer override of `pairing` ("per layer"), or None
    latent_dim: int = 512
    rope_dim: int = 64                  # rotated elements per head
    rope_heads: int = 1                 # heads in the rotated band (1 = MLA K_pe; kv_heads = full-width K)
    inv_freq: np.ndarray = None         # fp32 [rope_dim/2]
    # (request, start, end, repl_len, repl_row, semantic), sorted by (request, start)
    directives: list = field(default_factory=list)
    seed: int = 0
    pool_factor: float = 1.25           # pool pages = ceil(live pages * pool_factor) + extra_pages
    extra_pages: int = 0
    # filled by finalize()
    pt_offsets: np.ndarray = None       # int64 [n_req+1]
    pages: np.ndarray = None            # int32, concatenated page-table rows
    free_pages: np.ndarray = None       # int32, remaining pool pages in permuted order
    pool_pages: int = 0
    n_repl_rows: int = 0

    @property
    def elem_bytes(self):
        return 2 if self.dtype == DT_BF16 else 1

    @property
    def row_bytes(self):
        return self.row_elems * self.elem_bytes

    @property
    def row_elems(self):
        return self.latent_dim + self.rope_heads * self.rope_dim

    @property
    def n_slots(self):
        return self.pool_pages * self.page_size

    @property
    def layer_bytes(self):
        return self.n_slots * self.row_bytes

    @property
    def n_requests(self):
        return len(self.seq_lens)

    def pairing_of(self, layer: int) -> int:
        return self.pairing if self.layer_pairing is None else int(self.layer_pairing[layer])

    def free_slots(self) -> np.ndarray:
        """Token-level free slot ids (for ROTATE_ONLY): the slots of the free pages, in free-list order."""
        P = self.page_size
        return (self.free_pages.astype(np.int64)[:, None] * P + np.arange(P)[None, :]).reshape(-1).astype(np.int32)

    def finalize(self):
        """Page tables = a seeded random permutation of the pool's pages (so pages are NOT physically
        contiguous); free list = the remaining pages in permuted order."""
        P = self.page_size
        n_pages = [-(-int(L) // P) for L in self.seq_lens]
        live = sum(n_pages)
        self.pool_pages = int(math.ceil(live * self.pool_factor)) + int(self.extra_pages)
        rng = np.random.default_rng(self.seed + 7919)
        perm = rng.permutation(self.pool_pages).astype(np.int32)
        self.pt_offsets = np.zeros(len(n_pages) + 1, np.int64)
        self.pt_offsets[1:] = np.cumsum(n_pages)
        self.pages = perm[:live].copy()
        self.free_pages = perm[live:].copy()
        row = 0
        fixed = []
        for (r, s, e, n, _, sem) in self.directives:
            fixed.append((r, s, e, n, row, sem))
            row += n
        self.directives = fixed
        self.n_repl_rows = row
        return self


def fresh_pages_needed(w: Workload) -> int:
    """Upper bound on free pages a FRESH plan can consume: every request may be rewritten entirely,
    plus growth.  (Sizing only; the library and the oracle count the real number themselves.)"""
    P = w.page_size
    grow = sum(d[3] for d in w.directives)
    return sum(-(-int(L) // P) for L in w.seq_lens) + -(-grow // P) + w.n_requests


# ----------------------------------------------------------------------------- directive generators

def random_directives(rng: np.random.Generator, L: int, n: int, span_lo: int, span_hi: int, repl_hi: int,
                      log_uniform: bool = True, max_tries: int = 1000):
    """n sorted non-overlapping (start, end, repl_len) on a request of L tokens: start uniform, span length
    log-uniform (or uniform) in [span_lo, span_hi], replacement length uniform in [0, repl_hi]; the whole set is
    resampled on overlap (BASELINE.json config 4; edit shapes of PAPER.md:433-445)."""
    for _ in range(max_tries):
        out = []
        for _ in range(n):
            if log_uniform:
                ln = int(round(math.exp(rng.uniform(math.log(span_lo), math.log(span_hi)))))
            else:
                ln = int(rng.integers(span_lo, span_hi + 1))
            ln = max(0, min(ln, L))
            s = int(rng.integers(0, L - ln + 1))
            out.append((s, s + ln, int(rng.integers(0, repl_hi + 1))))
        out.sort()
        if all(out[i][0] >= out[i - 1][1] for i in range(1, len(out))):
            return out
    raise RuntimeError("could not place non-overlapping directives")


# ----------------------------------------------------------------------------- the five BASELINE.json configs

def config(n: int, **over) -> Workload:
    """BASELINE.json ``configs[n-1]`` (1-based like SURVEY.md section 8(d)); "3m" is the misaligned variant of 3.
    Span starts of configs 3/5 are not given by BASELINE.json; L/16, L/4, 3L/4 are this build's choice."""
    if n == 1:
        w = Workload("cfg1_2L_4K_p1", 2, [4096], 1, inv_freq=rope_inv_freq(64, 10000.0),
                     directives=[(0, 1000, 1600, 32, 0, AMORTIZE)], seed=0)
    elif n == 2:
        w = Workload("cfg2_dsv2lite_27L_32K", 27, [32768], 64, inv_freq=rope_inv_freq(64, 10000.0),
                     directives=[(0, 4096, 12288, 128, 0, AMORTIZE)], seed=0)
    elif n in (3, "3m"):
        L = 131072
        repl = (64, 0, 256) if n == 3 else (67, 3, 251)
        w = Workload("cfg3_dsv3_61L_128K" if n == 3 else "cfg3m_dsv3_61L_128K_misaligned", 61, [L], 64,
                     inv_freq=yarn_inv_freq(64, 10000.0, 40.0, 4096),
                     directives=[(0, L // 16, L // 16 + 2048, repl[0], 0, AMORTIZE),
                                 (0, L // 4, L // 4 + 16384, repl[1], 0, AMORTIZE),
                                 (0, 3 * L // 4, 3 * L // 4 + 512, repl[2], 0, AMORTIZE)], seed=0)
    elif n == 4:
        rng = np.random.default_rng(4)
        n_req, L = 64, 16384
        dirs = []
        for r in range(n_req):
            k = int(rng.integers(1, 5))
            for (s, e, rl) in random_directives(rng, L, k, 64, 4096, 256):
                dirs.append((r, s, e, rl, 0, AMORTIZE))
        w = Workload("cfg4_batched_64x16K_61L", 61, [L] * n_req, 64, inv_freq=yarn_inv_freq(64, 10000.0, 40.0, 4096),
                     directives=dirs, seed=4)
    elif n == 5:
        n_req, L = 8, 65536
        dirs = []
        for r in range(n_req):
            dirs += [(r, L // 16, L // 16 + 2048, 64, 0, AMORTIZE), (r, L // 4, L // 4 + 16384, 0, 0, AMORTIZE),
                     (r, 3 * L // 4, 3 * L // 4 + 512, 256, 0, AMORTIZE)]
        w = Workload("cfg5_fp8_8x64K_61L", 61, [L] * n_req, 64, dtype=DT_FP8,
                     inv_freq=yarn_inv_freq(64, 10000.0, 40.0, 4096), directives=dirs, seed=5)
    elif n == "gqa":
        # full-width K rotation.  K pool of a Llama-3.1-8B-style GQA model:
        # 32 layers, 8 kv heads x head_dim 128 (2048-B bf16 rows, all of it rotated), rope_theta 5e5 (Table 8 row 3,
        # PAPER.md:537), NeoX pairing, one request of 128K tokens, config 3's three directives.  V is position-free
        # and would be spliced as a latent-only pool with the same plan; it is not part of this workload.
        L = 131072
        w = Workload("gqa_llama31_32L_128K_8x128", 32, [L], 64, latent_dim=0, rope_dim=128, rope_heads=8,
                     inv_freq=rope_inv_freq(128, 5.0e5),
                     directives=[(0, L // 16, L // 16 + 2048, 64, 0, AMORTIZE),
                                 (0, L // 4, L // 4 + 16384, 0, 0, AMORTIZE),
                                 (0, 3 * L // 4, 3 * L // 4 + 512, 256, 0, AMORTIZE)], seed=6)
    elif n == "mha96":
        # Phi-3-style MHA K pool: 32 heads x head_dim 96 (12 chunks per head: not a power of two), theta 1e4
        # (Table 8 row 5), 32 layers x 32K tokens, misaligned replacements
        L = 32768
        w = Workload("mha_phi3_32L_32K_32x96", 32, [L], 64, latent_dim=0, rope_dim=96, rope_heads=32,
                     inv_freq=rope_inv_freq(96, 1.0e4),
                     directives=[(0, L // 16, L // 16 + 2048, 67, 0, AMORTIZE),
                                 (0, L // 4, L // 4 + 4096, 3, 0, AMORTIZE),
                                 (0, 3 * L // 4, 3 * L // 4 + 512, 251, 0, AMORTIZE)], seed=7)
    elif n == "appB":
        # The shape of the paper's own splice counters (App. B): DeepSeek-V2-Lite (27 layers, bf16,
        # token-level slots as in SGLang's pool), one run = 167-203 chunks spliced and ">= 740 MB rotated", i.e. ~129
        # tokens of 31,104 B per chunk.  Here: 185 chunk copies in ONE call.  Request k holds the d_k tokens in front of
        # a matched chunk plus its n_k tokens; the directive drops the d_k tokens, so the chunk lands in fresh slots
        # d_k positions earlier, rotated by -d_k (the paper's copy-to-dst_slots path).  n_k ~ U[66,194],
        # d_k ~ U[1,512] (the delta range of App. F); slots are a random permutation (worst case).
        rng = np.random.default_rng(383)
        n_req = 185
        n_k = rng.integers(66, 195, size=n_req)
        d_k = rng.integers(1, 513, size=n_req)
        w = Workload("appB_dsv2lite_185_chunks", 27, [int(a + b) for a, b in zip(d_k, n_k)], 1,
                     inv_freq=rope_inv_freq(64, 10000.0),
                     directives=[(r, 0, int(d_k[r]), 0, 0, AMORTIZE) for r in range(n_req)], seed=383)
    else:
        raise ValueError(n)
    for k, v in over.items():
        setattr(w, k, v)
    return w.finalize()


def scaled(w: Workload, n_layers: int | None = None) -> Workload:
    """Same workload with fewer layers (layers are independent buffers under one plan; used for parity samples)."""
    import copy
    v = copy.copy(w)
    if n_layers is not None:
        v.n_layers = n_layers
    return v


# ----------------------------------------------------------------------------- cache / replacement bytes

def fill_layer_(buf, w: Workload, layer: int, seed_base: int | None = None):
    """Fill one layer's pool (a torch uint8 tensor of w.layer_bytes bytes, any device) with N(0,1) values,
    seed = seed_base + layer, in the cache's storage type.  Returns the per-layer fp32 scale (1.0 for bf16;
    amax/448 for fp8 -- BASELINE.json config 5)."""
    import torch
    seed = (w.seed if seed_base is None else seed_base) * 1000003 + layer
    g = torch.Generator(device=buf.device)
    g.manual_seed(seed)
    n_elem = w.n_slots * w.row_elems
    if w.dtype == DT_BF16:
        view = buf.view(torch.bfloat16)
        assert view.numel() == n_elem
        view.normal_(0.0, 1.0, generator=g)
        return 1.0
    x = torch.empty(n_elem, dtype=torch.float32, device=buf.device)
    x.normal_(0.0, 1.0, generator=g)
    scale = torch.tensor(float(x.abs().max()) / 448.0, dtype=torch.float32).item()
    q = (x / scale).clamp_(-448.0, 448.0).to(torch.float8_e4m3fn)
    buf.copy_(q.view(torch.uint8))
    return scale


def fill_repl_(buf, w: Workload, layer: int, scale: float = 1.0):
    """Replacement rows of one layer (torch uint8 tensor of n_repl_rows * row_bytes), N(0,1), seed 1-based stream."""
    import torch
    if buf.numel() == 0:
        return
    g = torch.Generator(device=buf.device)
    g.manual_seed(1 * 1000003 + 7 * layer + 1 + w.seed * 31)
    n_elem = w.n_repl_rows * w.row_elems
    if w.dtype == DT_BF16:
        buf.view(torch.bfloat16).normal_(0.0, 1.0, generator=g)
        return
    x = torch.empty(n_elem, dtype=torch.float32, device=buf.device)
    x.normal_(0.0, 1.0, generator=g)
    q = (x / scale).clamp_(-448.0, 448.0).to(torch.float8_e4m3fn)
    buf.copy_(q.view(torch.uint8))
