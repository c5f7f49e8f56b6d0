"""Counter-based synthetic tensors for the MosaicQuant hot path.

Every value is a pure function of (seed, tensor_id, linear index): splitmix64 ->
two uniforms -> Box-Muller, so any slice can be regenerated independently and the
result does not depend on chunking or thread count.

The tensors stand in for the LLaMA3 / Qwen3 linear layers the paper measures on
(Table 5): dense Gaussian inliers plus rare large
outliers clustered in 64x64 blocks of the weight (Fig. 2a) and in
a few activation channels.  None of the method's arithmetic
lives here.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Dict, List, Tuple

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = 0x9E3779B97F4A7C15

# tensor ids
TID_W = 1
TID_A = 2
TID_XCAL = 3
TID_WBLK = 4
TID_WPOS = 5
TID_CH = 6


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        z = x + np.uint64(_GOLD)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def _key(seed: int, tensor_id: int, extra: int = 0) -> np.uint64:
    k = (seed * _GOLD + tensor_id * 0xD1B54A32D192ED03 + extra * 0x8CB92BA72F3D8DD7) & 0xFFFFFFFFFFFFFFFF
    return _splitmix64(np.array([k], dtype=np.uint64))[0]


def _hash_idx(key: np.uint64, idx: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        return _splitmix64(idx.astype(np.uint64) + key)


def _normal(key: np.uint64, start: int, count: int) -> np.ndarray:
    """count standard normals for linear indices [start, start+count) as float64."""
    idx = np.arange(start, start + count, dtype=np.uint64)
    with np.errstate(over="ignore"):
        x0 = _splitmix64(idx * np.uint64(2) + key)
        x1 = _splitmix64(idx * np.uint64(2) + np.uint64(1) + key)
    u1 = ((x0 >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)
    u2 = ((x1 >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def _normal_matrix(key: np.uint64, rows: int, cols: int, scale: float, chunk_rows: int = 0) -> np.ndarray:
    out = np.empty((rows, cols), dtype=np.float32)
    if chunk_rows <= 0:
        chunk_rows = max(1, (1 << 22) // max(cols, 1))
    for r0 in range(0, rows, chunk_rows):
        r1 = min(rows, r0 + chunk_rows)
        z = _normal(key, r0 * cols, (r1 - r0) * cols)
        out[r0:r1] = (scale * z).reshape(r1 - r0, cols).astype(np.float32)
    return out


def _smallest(key: np.uint64, n: int, count: int) -> np.ndarray:
    """`count` distinct indices in [0,n): those with the smallest hash (sorted ascending)."""
    h = _hash_idx(key, np.arange(n, dtype=np.uint64))
    if count >= n:
        return np.arange(n, dtype=np.int64)
    sel = np.argpartition(h, count)[:count]
    return np.sort(sel).astype(np.int64)


def outlier_channels(seed: int, K: int, exact: int | None = None) -> np.ndarray:
    """Outlier input-channel set C: chosen once per (seed, K); shared by A and X_cal."""
    cnt = exact if exact is not None else max(2, int(round(0.001 * K)))
    return _smallest(_key(seed, TID_CH, K), K, cnt)


def gen_weight(seed: int, N: int, K: int, sigma: float = 0.02, outlier_frac: float = 0.005,
               outlier_mult: float = 20.0) -> np.ndarray:
    """W[N,K] fp32 ~ N(0, sigma^2) with `outlier_frac` of entries x`outlier_mult`,
    clustered in 64x64 blocks (5% of the 64x64 blocks, at least 2)."""
    assert N % 64 == 0 and K % 64 == 0
    W = _normal_matrix(_key(seed, TID_W), N, K, sigma)
    nbn, nbk = N // 64, K // 64
    n_blocks = nbn * nbk
    n_ob = max(2, int(round(0.05 * n_blocks)))
    n_ob = min(n_ob, n_blocks)
    cnt = int(round(outlier_frac * N * K / n_ob))
    cnt = min(cnt, 4096)
    blocks = _smallest(_key(seed, TID_WBLK), n_blocks, n_ob)
    for b in blocks:
        bn, bk = divmod(int(b), nbk)
        pos = _smallest(_key(seed, TID_WPOS, int(b)), 4096, cnt)
        r, c = np.divmod(pos, 64)
        W[bn * 64 + r, bk * 64 + c] *= np.float32(outlier_mult)
    return W


def _act_f32(seed: int, tid: int, M: int, K: int, n_outlier_ch: int | None, mult: float) -> np.ndarray:
    A = _normal_matrix(_key(seed, tid), M, K, 1.0)
    C = outlier_channels(seed, K, n_outlier_ch)
    A[:, C] *= np.float32(mult)
    return A


def gen_act(seed: int, M: int, K: int, n_outlier_ch: int | None = None, mult: float = 10.0,
            dtype: str = "f16") -> np.ndarray:
    """A[M,K] ~ N(0,1) with the outlier channel set x`mult`.  dtype 'f16' -> np.float16 (RNE);
    'f32' -> the fp32 values before the 16-bit cast (the caller casts, e.g. to bf16)."""
    A = _act_f32(seed, TID_A, M, K, n_outlier_ch, mult)
    if dtype == "f16":
        return A.astype(np.float16)
    if dtype == "f32":
        return A
    raise ValueError(dtype)


def gen_calib(seed: int, K: int, n_tokens: int = 256, n_outlier_ch: int | None = None,
              mult: float = 10.0) -> np.ndarray:
    """X_cal[n_tokens,K] fp32: same law and same outlier channels as A, different tensor id."""
    return _act_f32(seed, TID_XCAL, n_tokens, K, n_outlier_ch, mult)


def budget_from_density(rho: float, N: int, K: int, block: int) -> int:
    """budget = floor(rho * n_blocks + 0.5) (reading A6)."""
    n_blocks = (N // block) * (K // block)
    return int(np.floor(rho * n_blocks + 0.5))


@dataclass(frozen=True)
class LayerShape:
    name: str
    K: int
    N: int


def _proj(hidden: int, inter: int, q_heads: int, kv_heads: int, head_dim: int = 128) -> List[LayerShape]:
    qkv = (q_heads + 2 * kv_heads) * head_dim
    return [
        LayerShape("qkv", hidden, qkv),
        LayerShape("o", q_heads * head_dim, hidden),
        LayerShape("gate_up", hidden, 2 * inter),
        LayerShape("down", inter, hidden),
    ]


# BASELINE.json `configs`, restated.  Shapes are LLaMA3 / Qwen3 projection sizes.
CONFIGS: Dict[str, dict] = {
    "tiny": dict(index=0, Ms=[16], layers=[LayerShape("tiny", 256, 256)], rho=2 / 16, block=64, seed=0),
    "llama3_8b_decode": dict(index=1, Ms=[1, 8, 32], layers=_proj(4096, 14336, 32, 8), rho=0.05, block=64, seed=1000),
    "llama3_8b_prefill": dict(index=2, Ms=[512, 2048, 8192], layers=_proj(4096, 14336, 32, 8), rho=0.05, block=64, seed=2000),
    "qwen3_8b": dict(index=3, Ms=[1, 128, 4096], layers=_proj(4096, 12288, 32, 8), rho=0.05, block=64, seed=3000,
                     rho_sweep=[0.0, 0.01, 0.05, 0.10], block_sweep=[64, 128]),
    "llama3_70b": dict(index=4, Ms=[1, 16, 4096], layers=_proj(8192, 28672, 64, 8), rho=0.05, block=64, seed=4000),
}


def config_shapes(name: str) -> List[Tuple[int, LayerShape]]:
    cfg = CONFIGS[name]
    return [(m, l) for m in cfg["Ms"] for l in cfg["layers"]]
