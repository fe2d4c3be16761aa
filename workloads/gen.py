"""Deterministic, position-addressable input bytes (same result on CPU and CUDA).

Every value is a pure function of ``(seed, stream, index)`` built from 64-bit
integer torch ops (wrap-around multiply, xor, shift), so a slab filled on the GPU
at full size can be re-derived byte-for-byte on the host for any sampled offset.
No arithmetic of the method lives here.
"""
from __future__ import annotations

import math
from typing import Tuple

import numpy as np
import torch

SEED0 = 25111617  # arxiv id; per-config seeds are SEED0 + 1000 * config index

_M64 = (1 << 64) - 1


def _s64(c: int) -> int:
    c &= _M64
    return c - (1 << 64) if c >= (1 << 63) else c


_GOLD = _s64(0x9E3779B97F4A7C15)
_C1 = _s64(0xBF58476D1CE4E5B9)
_C2 = _s64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    return (x >> k) & ((1 << (64 - k)) - 1)


def hash64(idx: torch.Tensor, seed: int, stream: int) -> torch.Tensor:
    """splitmix64 finaliser of (idx + key(seed, stream)); int64 in, int64 out (bit pattern)."""
    key = _s64((seed * 0x2545F4914F6CDD1D + (stream + 1) * 0xD6E8FEB86659FD93) & _M64)
    z = idx * _GOLD + key
    z = (z ^ _lsr(z, 30)) * _C1
    z = (z ^ _lsr(z, 27)) * _C2
    return z ^ _lsr(z, 31)


_CHUNK = 1 << 24


def fill_bytes(seed: int, stream: int, byte_offset: int, n_bytes: int, device="cpu",
               out: torch.Tensor | None = None) -> torch.Tensor:
    """uint8[n_bytes] = little-endian bytes of hash64(word index); offsets/sizes multiples of 8."""
    assert byte_offset % 8 == 0 and n_bytes % 8 == 0
    if out is None:
        out = torch.empty(n_bytes, dtype=torch.uint8, device=device)
    w = out.view(torch.int64)
    w0, nw = byte_offset // 8, n_bytes // 8
    for a in range(0, nw, _CHUNK):
        b = min(nw, a + _CHUNK)
        idx = torch.arange(w0 + a, w0 + b, dtype=torch.int64, device=out.device)
        w[a:b] = hash64(idx, seed, stream)
    return out


_IH_MEAN = 4 * 65535 / 2.0
_IH_STD = math.sqrt(4 * (65536.0 ** 2 - 1) / 12.0)


def normal16_at(idx: torch.Tensor, seed: int, stream: int, std: float, dtype: torch.dtype) -> torch.Tensor:
    """Value of the 16-bit N(0, std) stream at arbitrary int64 element indices (any shape)."""
    scale = np.float32(std / _IH_STD)
    h = hash64(idx, seed, stream)
    s = (h & 0xFFFF) + (_lsr(h, 16) & 0xFFFF) + (_lsr(h, 32) & 0xFFFF) + (_lsr(h, 48) & 0xFFFF)
    v = (s.to(torch.float32) - np.float32(_IH_MEAN)) * float(scale)
    return v.to(dtype)


def fill_normal16(seed: int, stream: int, elem_offset: int, n: int, std: float, dtype: torch.dtype,
                  device="cpu", out: torch.Tensor | None = None) -> torch.Tensor:
    """16-bit float tensor, approximately N(0, std): sum of the four 16-bit fields of hash64(index)
    (Irwin-Hall, 4 terms), centred, scaled in fp32, rounded once to ``dtype``."""
    assert dtype in (torch.float16, torch.bfloat16)
    if out is None:
        out = torch.empty(n, dtype=dtype, device=device)
    for a in range(0, n, _CHUNK):
        b = min(n, a + _CHUNK)
        idx = torch.arange(elem_offset + a, elem_offset + b, dtype=torch.int64, device=out.device)
        out[a:b] = normal16_at(idx, seed, stream, std, dtype)
    return out


def fill_kv_pool(pool: torch.Tensor, rows: int, heads_in_pool: int, dim: int, slot0: int, head0: int, n: int,
                 n_kv_heads: int, seed: int, stream: int, dtype: torch.dtype, row_chunk: int = 1 << 16,
                 layout: int = 0, block_size: int = 1) -> None:
    """Paged-KV content that is a pure function of (row, head, d): element d of KV head ``h`` at pool row ``row``
    (row = flattened (layer, K|V, block, token)) has the value of stream index (row * n_kv_heads + h) * dim + d,
    N(0,1).  Writes heads head0..head0+n-1 into slots slot0..slot0+n-1 of ``pool``; every other slot is left as it is.
    ``layout`` 0: pool viewed as [rows][heads_in_pool][dim] (token-major); ``layout`` 1: [rows / block_size][heads_in_pool]
    [block_size][dim] (head-major: the tokens of a block are contiguous per head).  Same values either way."""
    d = torch.arange(dim, dtype=torch.int64, device=pool.device)
    hh = torch.arange(head0, head0 + n, dtype=torch.int64, device=pool.device)
    if layout == 0:
        v = pool.view(dtype).view(rows, heads_in_pool, dim)
    else:
        assert rows % block_size == 0
        row_chunk = max(row_chunk // block_size, 1) * block_size
        v = pool.view(dtype).view(rows // block_size, heads_in_pool, block_size, dim)
    for a in range(0, rows, row_chunk):
        b = min(rows, a + row_chunk)
        r = torch.arange(a, b, dtype=torch.int64, device=pool.device)
        idx = ((r[:, None, None] * n_kv_heads + hh[None, :, None]) * dim) + d[None, None, :]
        val = normal16_at(idx, seed, stream, 1.0, dtype)                     # [rows of the chunk][n heads][dim]
        if layout == 0:
            v[a:b, slot0:slot0 + n, :] = val
        else:
            v[a // block_size:b // block_size, slot0:slot0 + n] = val.view((b - a) // block_size, block_size, n, dim).permute(0, 2, 1, 3)


def torch_dtype(name: str) -> torch.dtype:
    return {"bf16": torch.bfloat16, "fp16": torch.float16}[name]


def as_u8(t: torch.Tensor) -> np.ndarray:
    """CPU tensor -> numpy uint8 view of its bytes (bf16 has no numpy dtype)."""
    return t.detach().cpu().contiguous().view(torch.uint8).numpy()


def make_page_table(n_seqs: int, seq_lens, block_size: int, pool_slack: float, seed: int
                    ) -> Tuple[np.ndarray, np.ndarray, np.ndarray, int]:
    """Fragmented paged-KV bookkeeping: physical block ids are a seeded random subset/permutation
    of a pool of ceil(slack * live) blocks; ``last_use`` is a seeded permutation of 0..n_seqs-1.
    Returns (table[n_seqs][max_blocks] int32 with -1 = none, seq_lens int32, last_use int64, n_blocks)."""
    seq_lens = np.asarray(seq_lens, dtype=np.int32)
    assert seq_lens.shape == (n_seqs,)
    per = (seq_lens + block_size - 1) // block_size
    live = int(per.sum())
    n_blocks = int(math.ceil(pool_slack * live))
    max_blocks = int(per.max()) if n_seqs else 0
    rng = np.random.default_rng(seed)
    ids = rng.permutation(n_blocks)[:live].astype(np.int32)
    table = np.full((n_seqs, max_blocks), -1, dtype=np.int32)
    k = 0
    for s in range(n_seqs):
        table[s, : per[s]] = ids[k : k + per[s]]
        k += per[s]
    last_use = rng.permutation(n_seqs).astype(np.int64)
    return table, seq_lens, last_use, n_blocks


def microbench_intervals(n: int, lo: int, hi: int, seed: int, src_arena: int, max_total: int = 32 << 30):
    """Config 5b recipe: n intervals, size = 16*floor(exp(U(ln lo, ln hi))/16), random 16-B aligned
    source offsets in a ``src_arena``-byte arena (sources may overlap), destinations disjoint, laid out in
    random order with random 16-B aligned gaps (0..240 B).  Returns (src_off, dst_off, size, dst_arena)."""
    rng = np.random.default_rng(seed)
    size = (np.exp(rng.uniform(math.log(lo), math.log(hi), n)) // 16).astype(np.int64) * 16
    size = np.maximum(size, 16)
    tot = int(size.sum())
    if tot > max_total:          # clip the largest draws until the total fits
        size = np.minimum(size, max(16, (max_total // n) // 16 * 16 * 4))
    src_off = (rng.integers(0, max(1, (src_arena - int(size.max())) // 16), n)).astype(np.int64) * 16
    order = rng.permutation(n)
    gaps = rng.integers(0, 16, n).astype(np.int64) * 16
    dst_off = np.empty(n, dtype=np.int64)
    ends = np.cumsum(gaps[order] + size[order])
    dst_off[order] = ends - size[order]
    return src_off, dst_off, size, int(ends[-1]) if n else 0
