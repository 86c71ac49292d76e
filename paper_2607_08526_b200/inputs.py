"""Seeded synthetic inputs for configs C1-C5 (BASELINE.json `configs`).

This module is the ONLY thing the CUDA path's callers and the CPU oracle's
callers share.  It holds none of the method's arithmetic: it draws N(0, std)
tensors with numpy's counter-based generator and, where a config says bf16,
rounds the fp32 draw to bf16 with torch's library conversion.  Recipe (DESIGN.md
"Input recipe", reading R15): `numpy.random.default_rng([0, config_id,
tensor_id])`, fp32 standard-normal draw times std, then RNE to bf16.

No dataset or benchmark suite is involved; the shapes stand in for the medium
Stable Audio 3 DiT (24 blocks, d_model 1536 -- PAPER.md L47, L142).
"""
from __future__ import annotations

import numpy as np
import torch

D_MODEL = 1536            # PAPER.md L47 / L142 (medium)
N_BLOCKS = 24             # PAPER.md L47 / L142
D_QKV = 3 * D_MODEL       # fused QKV (config C2)
D_MLP = 4 * D_MODEL       # config C3: 1536 -> 6144 -> 1536
W_STD = 0.02              # reading R5: 0.02 is a standard deviation
B_STD = 0.01              # config C1
OUTLIER_FRAC = 0.01       # config C3: "1% of K channels scaled x20"
OUTLIER_GAIN = 20.0

# The paper's two released DiT sizes: (d_model, blocks).
MODELS = {"medium": (1536, 24), "small-music": (1024, 20)}
SAMPLING_STEPS = 8        # 8 denoising steps per clip ("fast preset" 6, L222)


def block_linears(d_model: int = D_MODEL):
    """(name, K, N, activation-after) of one DiT block's linears, config C5 order (fused QKV, MLP ratio 4)."""
    return (("qkv", d_model, 3 * d_model, "none"), ("out", d_model, d_model, "none"),
            ("up", d_model, 4 * d_model, "gelu"), ("down", 4 * d_model, d_model, "none"))


BLOCK_LINEARS = block_linears(D_MODEL)


def normal_f32(shape, std: float, config_id: int, tensor_id: int) -> np.ndarray:
    rng = np.random.default_rng([0, int(config_id), int(tensor_id)])
    x = rng.standard_normal(size=shape, dtype=np.float32)
    return (x * np.float32(std)).astype(np.float32)


def bf16_bits(x_f32: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit patterns (uint16), round-to-nearest-even (torch)."""
    t = torch.from_numpy(np.ascontiguousarray(x_f32, dtype=np.float32)).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16).copy()


def bf16_as_f32(bits: np.ndarray) -> np.ndarray:
    """bf16 bit patterns -> the same values widened (exactly) to fp32."""
    return (np.asarray(bits, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32)


def normal_bf16(shape, std: float, config_id: int, tensor_id: int):
    """Returns (bits uint16, values fp32) of a bf16 N(0,std) tensor."""
    b = bf16_bits(normal_f32(shape, std, config_id, tensor_id))
    return b, bf16_as_f32(b)


def outlier_channels(K: int, config_id: int, tensor_id: int) -> np.ndarray:
    """Reading R13: round(0.01*K) fixed channels, seeded, same for every token."""
    n = int(round(OUTLIER_FRAC * K))
    rng = np.random.default_rng([0, int(config_id), int(tensor_id)])
    return np.sort(rng.choice(K, size=n, replace=False))


def c1():
    """C1 W8A8 tiny, all fp32, 'seed 0'."""
    return {"X": normal_f32((64, 256), 1.0, 1, 0), "W": normal_f32((256, 256), W_STD, 1, 1),
            "b": normal_f32((256,), B_STD, 1, 2)}


def c2(M: int = 512):
    """C2 attention projections: bf16 X [M,1536], Wqkv [4608,1536], Wout [1536,1536], bf16 bias."""
    Xb, X = normal_bf16((M, D_MODEL), 1.0, 2, 0)
    return {"X_bits": Xb, "X": X,
            "Wqkv": normal_f32((D_QKV, D_MODEL), W_STD, 2, 1),
            "Wout": normal_f32((D_MODEL, D_MODEL), W_STD, 2, 2),
            "bqkv": normal_bf16((D_QKV,), B_STD, 2, 3), "bout": normal_bf16((D_MODEL,), B_STD, 2, 4)}


def c3(M: int = 4096, K: int = D_MODEL, H: int = D_MLP):
    """C3 MLP with outlier activations: X bf16 [M,K] with 1% channels x20; Wup [H,K], Wdown [K,H]."""
    x = normal_f32((M, K), 1.0, 3, 0)
    ch = outlier_channels(K, 3, 5)
    x[:, ch] *= np.float32(OUTLIER_GAIN)
    Xb = bf16_bits(x)
    return {"X_bits": Xb, "X": bf16_as_f32(Xb), "outlier_channels": ch,
            "Wup": normal_f32((H, K), W_STD, 3, 1), "Wdown": normal_f32((K, H), W_STD, 3, 2),
            "bup": normal_bf16((H,), B_STD, 3, 3), "bdown": normal_bf16((K,), B_STD, 3, 4)}


C4_SHAPES = ((D_MODEL, D_QKV), (D_MODEL, D_MLP), (D_MLP, D_MODEL))  # (K, N)
C4_MS = (32, 512, 4096)


def c4(M: int, K: int, N: int):
    """C4 W4A16: bf16 X [M,K], W fp32 [N,K] (to be int4-g32 quantised), bf16 bias."""
    tid = (M * 7 + K * 3 + N) % 100000
    Xb, X = normal_bf16((M, K), 1.0, 4, tid)
    return {"X_bits": Xb, "X": X, "W": normal_f32((N, K), W_STD, 4, tid + 100000),
            "b": normal_bf16((N,), B_STD, 4, tid + 200000)}


def c5_layer(block: int, which: int, M: int = 2048, d_model: int = D_MODEL):
    """C5: linear `which` (index into block_linears) of block `block`: own N(0,1)
    bf16 input (reading R14), W ~N(0,0.02), bf16 bias.  d_model = 1024 gives the small-music
    shapes (NEXT-4), drawn from config id 6 so that the medium tensors keep their seeds."""
    name, K, N, act = block_linears(d_model)[which]
    cid = 5 if d_model == D_MODEL else 6
    tid = block * 16 + which * 4
    Xb, X = normal_bf16((M, K), 1.0, cid, tid)
    return {"name": name, "K": K, "N": N, "act": act, "X_bits": Xb, "X": X,
            "W": normal_f32((N, K), W_STD, cid, tid + 1), "b": normal_bf16((N,), B_STD, cid, tid + 2)}


def steer_direction(d_model: int, tensor_id: int = 0):
    """A seeded unit direction d (fp32, eq. 1's normalisation applied in fp64) standing in for a
    difference-in-means direction, and a baseline residual norm ||h-bar|| of the magnitude a N(0,1)
    residual row has (sqrt(d_model))."""
    rng = np.random.default_rng([0, 7, int(tensor_id)])
    v = rng.standard_normal(d_model)
    return (v / np.linalg.norm(v)).astype(np.float32), float(np.sqrt(d_model))


HEAD_DIM = 64             # reading R21: d_model / 64 heads (24 for medium, 16 for small-music)


def norm_params(K: int, tensor_id: int = 0):
    """Seeded LayerNorm / RMSNorm parameters (fp32): gain ~ 1 + 0.1 N(0,1), shift ~ 0.05 N(0,1)."""
    g = (1.0 + normal_f32((K,), 0.1, 8, 2 * tensor_id)).astype(np.float32)
    b = normal_f32((K,), 0.05, 8, 2 * tensor_id + 1)
    return g, b


def residual_stream(M: int, K: int, tensor_id: int = 0, outliers: bool = True, mean: float = 0.25):
    """A bf16 residual-stream tensor [M,K] ~ N(mean, 1) with C3-style outlier channels (1% of K, x20): what the
    block's normalisation sees.  Returns (bits, fp32 values)."""
    x = normal_f32((M, K), 1.0, 8, 100 + tensor_id) + np.float32(mean)
    if outliers:
        x[:, outlier_channels(K, 8, 200 + tensor_id)] *= np.float32(OUTLIER_GAIN)
    b = bf16_bits(x)
    return b, bf16_as_f32(b)


def qkv_activations(B: int, S: int, H: int, Dh: int = HEAD_DIM, tensor_id: int = 0, q_gain: float = 1.0):
    """bf16 [B*S, 3*H*Dh] ~ N(0,1) standing in for the fused QKV projection's output (columns [q | k | v]);
    q_gain > 1 sharpens the softmax.  Returns (bits, fp32 values)."""
    x = normal_f32((B * S, 3 * H * Dh), 1.0, 8, 300 + tensor_id)
    x[:, : H * Dh] *= np.float32(q_gain)
    b = bf16_bits(x)
    return b, bf16_as_f32(b)
