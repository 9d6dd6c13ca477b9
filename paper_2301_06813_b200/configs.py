"""Seeded synthetic inputs for the five BASELINE.json configs ("Input recipe").

This module holds NO arithmetic of the method (no cost formula, no DP, no CD): it only
describes layer lists, meshes and network parameters as plain numpy records, and draws the
random shapes / Coordinate Descent starts from splitmix64.  It is the one module that both the
CUDA path (paper_2301_06813_b200.binding) and the test oracle (oracle/ref.py) are fed from.

The paper's own workloads (VGG13 / GPT layer lists, fitted alpha-beta of Piz Daint and Google
Cloud) are not available; these inputs take their shapes from
BASELINE.json's configs and stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

# 64-byte layer record, identical byte layout to `autoddl_layer` (include/autoddl.h)
LAYER_DTYPE = np.dtype(
    [
        ("M", "<i8"), ("Kd", "<i8"), ("N", "<i8"),
        ("in_rows", "<i8"), ("in_cols", "<i8"),
        ("kind", "<i4"), ("act_bytes", "<i4"), ("wgrad_bytes", "<i4"),
        ("wstate_bytes", "<i4"), ("max_split_rows", "<i4"), ("max_split_cols", "<i4"),
    ],
    align=False,
)
assert LAYER_DTYPE.itemsize == 64

GEMM, ATTN = 0, 1
INTRA, INTER = 0, 1
FOLD = 0x4000            # bit 14 of mesh.link[0]: the folded factorisation space (R28)

# picoseconds; 5 us intra-node, 20 us inter-node (BASELINE.json configs[0])
ALPHA_PS = (5_000_000, 20_000_000)
# integer ps/byte: 300 GB/s -> 3 (reading R3/A7), 25 GB/s -> 40, 12.5 GB/s -> 80
BETA_300, BETA_25, BETA_12_5 = 3, 40, 80

_MASK64 = (1 << 64) - 1


class SplitMix64:
    """splitmix64; first output for seed 0 is 0xE220A8397B1DCDAF."""

    def __init__(self, seed: int):
        self.state = seed & _MASK64

    def next(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & _MASK64
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK64
        return z ^ (z >> 31)

    def next_array(self, n: int) -> np.ndarray:
        """n consecutive outputs, vectorised (same sequence as n calls of next())."""
        with np.errstate(over="ignore"):
            idx = np.arange(1, n + 1, dtype=np.uint64)
            z = np.uint64(self.state) + idx * np.uint64(0x9E3779B97F4A7C15)
            self.state = int(z[-1]) if n else self.state
            z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
            z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
            return z ^ (z >> np.uint64(31))


@dataclass
class Mesh:
    size: tuple          # level 0 outermost
    link: tuple          # INTRA / INTER per level

    @property
    def ndim(self) -> int:
        return len(self.size)

    @property
    def K(self) -> int:
        """6^ndim for ndim <= 3; beyond, the signature index runs over the allowed rows only (R26); folded
        (bit 14 of link[0], R28): the product over the groups of equal levels of the number of ordered factorisations"""
        if self.link[0] & FOLD:
            k, d = 1, 0
            while d < self.ndim:
                n = 1
                while d + n < self.ndim and self.size[d + n] == self.size[d] and (self.link[d + n] & 1) == (self.link[d] & 1):
                    n += 1
                k *= (n + 2) * (n + 1) // 2
                d += n
            return k
        if self.ndim <= 3:
            return 6 ** self.ndim
        k = 1
        for l in self.link:
            a = (l >> 8) & 0x3F
            k *= bin(a).count("1") if a else 6
        return k


@dataclass
class Net:
    alpha_ps: tuple = ALPHA_PS               # (intra, inter)
    beta_ps_per_byte: tuple = (BETA_300, BETA_25)
    mem_cap_bytes: int = 0                   # 0 = no cap
    micro_batches: int = 1                   # gradient accumulation: redistributions per weight-gradient synchronisation


@dataclass
class Workload:
    name: str
    layers: np.ndarray                       # LAYER_DTYPE [Bp, L]
    mesh: Mesh
    net: Net
    S: int                                   # CD starts per problem
    seed: int = 0
    max_sweeps: int = 64
    extra: dict = field(default_factory=dict)

    @property
    def Bp(self) -> int:
        return self.layers.shape[0]

    @property
    def L(self) -> int:
        return self.layers.shape[1]

    @property
    def K(self) -> int:
        return self.mesh.K

    @property
    def cells(self) -> int:
        return self.Bp * self.L * self.K * self.K

    def cd_init(self) -> np.ndarray:
        """init[p][s][l] = next_B() % K in p-major, s, l order; stream B = seed + 1."""
        rng = SplitMix64(self.seed + 1)
        r = rng.next_array(self.Bp * self.S * self.L)
        return (r % np.uint64(self.K)).astype(np.int32).reshape(self.Bp, self.S, self.L)


def gemm(M, Kd, N, act, wgrad, wstate, in_rows=None, in_cols=None, max_rows=None, max_cols=None):
    rec = np.zeros((), dtype=LAYER_DTYPE)
    rec["M"], rec["Kd"], rec["N"] = M, Kd, N
    rec["in_rows"] = M if in_rows is None else in_rows
    rec["in_cols"] = Kd if in_cols is None else in_cols
    rec["kind"] = GEMM
    rec["act_bytes"], rec["wgrad_bytes"], rec["wstate_bytes"] = act, wgrad, wstate
    rec["max_split_rows"] = min(M if max_rows is None else max_rows, 2**31 - 1)
    rec["max_split_cols"] = min(N if max_cols is None else max_cols, 2**31 - 1)
    return rec


def attn(M, N, in_cols, act, max_rows, max_cols):
    rec = np.zeros((), dtype=LAYER_DTYPE)
    rec["M"], rec["Kd"], rec["N"] = M, 0, N
    rec["in_rows"], rec["in_cols"] = M, in_cols
    rec["kind"] = ATTN
    rec["act_bytes"], rec["wgrad_bytes"], rec["wstate_bytes"] = act, 0, 0
    rec["max_split_rows"], rec["max_split_cols"] = max_rows, max_cols
    return rec


def _stack(recs) -> np.ndarray:
    out = np.zeros((1, len(recs)), dtype=LAYER_DTYPE)
    for l, r in enumerate(recs):
        out[0, l] = r
    return out


def config1_tiny() -> Workload:
    """BASELINE.json configs[0]: 4 fp32 GEMMs 1024->1024, batch 32, mesh 2 nodes x 2 GPUs."""
    recs = [gemm(32, 1024, 1024, act=4, wgrad=4, wstate=8) for _ in range(4)]
    return Workload("tiny", _stack(recs), Mesh((2, 2), (INTER, INTRA)), Net(ALPHA_PS, (BETA_300, BETA_25), 0), S=16)


def config2_vgg16() -> Workload:
    """configs[1]: 13 convs as im2col GEMMs + 3 FC, fp32, batch 64, mesh 8 nodes x 1 GPU, 16 GB cap."""
    B = 64
    convs = [(3, 64, 224), (64, 64, 224), (64, 128, 112), (128, 128, 112), (128, 256, 56), (256, 256, 56),
             (256, 256, 56), (256, 512, 28), (512, 512, 28), (512, 512, 28), (512, 512, 14), (512, 512, 14),
             (512, 512, 14)]
    recs = [gemm(B * h * h, 9 * cin, cout, act=4, wgrad=4, wstate=12, in_rows=B * h * h, in_cols=cin)
            for (cin, cout, h) in convs]
    for (kd, n) in [(25088, 4096), (4096, 4096), (4096, 1000)]:
        recs.append(gemm(B, kd, n, act=4, wgrad=4, wstate=12))
    return Workload("vgg16", _stack(recs), Mesh((8, 1), (INTER, INTRA)),
                    Net(ALPHA_PS, (BETA_300, BETA_12_5), 16 * 10**9), S=64)


def _transformer_block(M, H, F, act, wgrad, wstate, attn_rows, attn_heads):
    return [
        gemm(M, H, 3 * H, act, wgrad, wstate),
        attn(M, H, 3 * H, act, attn_rows, attn_heads),
        gemm(M, H, H, act, wgrad, wstate),
        gemm(M, H, F, act, wgrad, wstate),
        gemm(M, F, H, act, wgrad, wstate),
    ]


def config3_transformer24() -> Workload:
    """configs[2]: 24 blocks (QKV, attention, out proj, MLP up, MLP down), fp16 act / fp32 grads, mesh 4 x 8."""
    M, H = 8 * 512, 1024
    recs = []
    for _ in range(24):
        recs += _transformer_block(M, H, 4096, act=2, wgrad=4, wstate=18, attn_rows=8, attn_heads=16)
    return Workload("transformer24", _stack(recs), Mesh((4, 8), (INTER, INTRA)),
                    Net(ALPHA_PS, (BETA_300, BETA_25), 40 * 10**9), S=256)


def _dims(r: np.ndarray) -> np.ndarray:
    """piecewise log-uniform on [256, 16256], multiples of 4"""
    base = np.uint64(64) + ((r >> np.uint64(8)) % np.uint64(64))
    return (base << ((r % np.uint64(6)) + np.uint64(2))).astype(np.int64)


def config4_batched(Bp: int = 4096, L: int = 64, seed: int = 0) -> Workload:
    """configs[3]: Bp independent chains of L GEMMs, dims log-uniform in [256, 16384], fp16, mesh 4 x 4."""
    rng = SplitMix64(seed)
    d = _dims(rng.next_array(Bp * (L + 2))).reshape(Bp, L + 2)   # per problem: M_p, d_0..d_L
    layers = np.zeros((Bp, L), dtype=LAYER_DTYPE)
    M = d[:, 0:1]
    layers["M"] = np.broadcast_to(M, (Bp, L))
    layers["Kd"] = d[:, 1:L + 1]
    layers["N"] = d[:, 2:L + 2]
    layers["in_rows"] = layers["M"]
    layers["in_cols"] = layers["Kd"]
    layers["kind"] = GEMM
    layers["act_bytes"], layers["wgrad_bytes"], layers["wstate_bytes"] = 2, 4, 18
    layers["max_split_rows"] = layers["M"]
    layers["max_split_cols"] = layers["N"]
    return Workload("batched", layers, Mesh((4, 4), (INTER, INTRA)), Net(ALPHA_PS, (BETA_300, BETA_25), 0),
                    S=1, seed=seed)


def config5_transformer96() -> Workload:
    """configs[4]: 96 blocks, hidden 12288, MLP 49152, 1024 token rows, mesh 8 x 8 x 8 (64 nodes x 8 GPUs), K=216."""
    M, H = 1024, 12288
    recs = []
    for _ in range(96):
        recs += _transformer_block(M, H, 49152, act=2, wgrad=4, wstate=18, attn_rows=1, attn_heads=96)
    return Workload("transformer96", _stack(recs), Mesh((8, 8, 8), (INTER, INTER, INTRA)),
                    Net(ALPHA_PS, (BETA_300, BETA_25), 80 * 10**9), S=1024)


PAPER_ROWS = 0x07 << 8   # mesh.link bits 8..13: rows {0, 1, 2} = the paper's SBP matmul factors (R24)


def config6_paper_space(restricted: bool = True) -> Workload:
    """Not in BASELINE.json: the Transformer-24 chain on 4 nodes x 2 GPUs refined into prime sub-levels (2 . 2 | 2) with
    the matmul rows only -- the paper's own factorisation space: 27 of the 216 signatures."""
    M, H = 8 * 512, 1024
    recs = []
    for _ in range(24):
        recs += _transformer_block(M, H, 4096, act=2, wgrad=4, wstate=18, attn_rows=8, attn_heads=16)
    allow = PAPER_ROWS if restricted else 0
    return Workload("paper-space", _stack(recs), Mesh((2, 2, 2), (INTER | allow, INTER | allow, INTRA | allow)),
                    Net(ALPHA_PS, (BETA_300, BETA_25), 40 * 10**9), S=64)


def config7_two_nodes_sixteen_gpus() -> Workload:
    """Not in BASELINE.json: the paper's Google Cloud machine, 2 nodes x 16 GPUs refined into prime
    sub-levels 2 | 2.2.2.2, searched over the matmul rows {0,1,2} per sub-level (K = 3^5 = 243, R26), on the
    shape of the paper's large Transformer (28 layers, model dimension 4,096, 32 heads, 2,048 sequences of
    1,024 tokens per batch, run as 64 micro-batches of 32 sequences (PAPER.md:283 gradient accumulation, R25);
    synthetic records, no weights).  Data parallelism does not fit the 40 GB cap, as in the paper."""
    M, H = 32 * 1024, 4096
    recs = []
    for _ in range(28):
        recs += _transformer_block(M, H, 4 * H, act=2, wgrad=4, wstate=18, attn_rows=32, attn_heads=32)
    a = PAPER_ROWS
    return Workload("two-nodes-x-16-gpus", _stack(recs), Mesh((2, 2, 2, 2, 2), (INTER | a, INTRA | a, INTRA | a, INTRA | a, INTRA | a)),
                    Net(ALPHA_PS, (BETA_300, BETA_25), 40 * 10**9, micro_batches=64), S=64)


def config8_vgg13_32_nodes() -> Workload:
    """Not in BASELINE.json: the setting of the paper's Fig. 8: VGG13 on 32 single-GPU nodes of Piz Daint
    (batch = 8 x nodes, fp32, 16 GB), the nodes refined into prime sub-levels 2.2.2.2.2 and searched over
    the matmul rows (K = 243, R26).  Convolutions as im2col GEMMs as in config 2; synthetic records."""
    B = 8 * 32
    convs = [(3, 64, 224), (64, 64, 224), (64, 128, 112), (128, 128, 112), (128, 256, 56), (256, 256, 56),
             (256, 512, 28), (512, 512, 28), (512, 512, 14), (512, 512, 14)]
    recs = [gemm(B * h * h, 9 * cin, cout, act=4, wgrad=4, wstate=12, in_rows=B * h * h, in_cols=cin)
            for (cin, cout, h) in convs]
    for (kd, n) in [(25088, 4096), (4096, 4096), (4096, 1000)]:
        recs.append(gemm(B, kd, n, act=4, wgrad=4, wstate=12))
    return Workload("vgg13-32-nodes", _stack(recs), Mesh((2, 2, 2, 2, 2), (INTER | PAPER_ROWS,) * 5),
                    Net(ALPHA_PS, (BETA_300, BETA_12_5), 16 * 10**9), S=64)


def config9_piz_daint_transformer(nodes: int = 64) -> Workload:
    """Not in BASELINE.json: the paper's Piz Daint Transformer runs (model dimension 8,192, 64 heads of 128,
    8 / 20 / 44 layers on 64 / 128 / 256 single-GPU P100 nodes, batch 1,024 sequences of 1,024 tokens, fp32), searched in
    the FOLDED factorisation space (R28): the nodes as 6 / 7 / 8 equal prime sub-levels of size 2, one signature
    per ordered factorisation p = p0 p1 p2 (K = 28 / 36 / 45).  The batch runs as 256 micro-batches of 4 sequences
    (R25), which keeps a feasible strategy under the per-layer memory budget of R7 at every size.
    Synthetic records, no weights."""
    n = {64: 6, 128: 7, 256: 8}[nodes]
    layers = {64: 8, 128: 20, 256: 44}[nodes]
    M, H = 4 * 1024, 8192
    recs = []
    for _ in range(layers):
        recs += _transformer_block(M, H, 4 * H, act=4, wgrad=4, wstate=16, attn_rows=4, attn_heads=64)
    return Workload("piz-daint-transformer-%d-nodes" % nodes, _stack(recs), Mesh((2,) * n, (INTER | FOLD,) + (INTER,) * (n - 1)),
                    Net(ALPHA_PS, (BETA_300, BETA_12_5), 16 * 10**9, micro_batches=256), S=64)


CONFIGS = {
    1: config1_tiny,
    2: config2_vgg16,
    3: config3_transformer24,
    4: config4_batched,
    5: config5_transformer96,
    6: config6_paper_space,
    7: config7_two_nodes_sixteen_gpus,
    8: config8_vgg13_32_nodes,
    9: config9_piz_daint_transformer,
    10: lambda: config9_piz_daint_transformer(128),
    11: lambda: config9_piz_daint_transformer(256),
}
