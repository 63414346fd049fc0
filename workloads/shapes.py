"""Bucket layouts of the five BASELINE.json configs — shapes only.

This module holds NO arithmetic of the method (no routing, packing, counting or reducing):
it lists parameter tensors of the model families the paper's workloads use (PAPER.md L297,
Tables 3/4/13), marks which ones the binding makes low-bit candidates (PAPER L205, L215-217:
backbone / encoder weight matrices eligible; embeddings, norms, biases and heads FP32), and
splits them into DDP-style buckets: iterate tensors in REVERSE registration
order, never split a tensor, close the bucket once its cumulative size >= cap.
It serves both the oracle tests and the CUDA path's tests/bench as an input description.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Tuple


@dataclass(frozen=True)
class TensorSpec:
    name: str
    numel: int
    eligible: bool          # binding: low-bit candidate (True) or FP32-only (False)
    layer: int = -1         # transformer layer index (GPT sigma schedule), -1 otherwise


@dataclass
class Bucket:
    index: int
    tensors: List[TensorSpec]
    off: List[int] = field(default_factory=list)
    n: int = 0

    def __post_init__(self):
        o = 0
        self.off = []
        for t in self.tensors:
            self.off.append(o)
            o += t.numel
        self.n = o

    @property
    def length(self) -> List[int]:
        return [t.numel for t in self.tensors]

    @property
    def elig(self) -> List[int]:
        return [1 if t.eligible else 0 for t in self.tensors]

    @property
    def n_eligible(self) -> int:
        return sum(t.numel for t in self.tensors if t.eligible)


@dataclass
class Config:
    name: str
    index: int              # c = 0..4, the seed base
    W: int
    buckets: List[Bucket]
    dist: str               # "gauss" | "student3"
    sigma_lo: float         # per-tensor sigma ~ 10^U(log10 lo, log10 hi); ignored for "layer" schedule
    sigma_hi: float
    sigma_schedule: str     # "loguniform" | "gpt_layer" | "const"
    zero_frac: float        # fraction of positions forced to +0.0 (iid Bernoulli per worker)
    nan_frac: float = 0.0   # fraction of positions forced to NaN ...
    nan_bucket: int = -1    # ... in this bucket ...
    nan_worker: int = -1    # ... of this worker only

    @property
    def n_params(self) -> int:
        return sum(b.n for b in self.buckets)

    @property
    def n_tensors(self) -> int:
        return sum(len(b.tensors) for b in self.buckets)


def bucketize(tensors: List[TensorSpec], cap_elems: int) -> List[Bucket]:
    """DDP-style: reverse registration order, whole tensors, close when cumulative >= cap."""
    buckets: List[Bucket] = []
    cur: List[TensorSpec] = []
    size = 0
    for t in reversed(tensors):
        cur.append(t)
        size += t.numel
        if size >= cap_elems:
            buckets.append(Bucket(len(buckets), cur))
            cur, size = [], 0
    if cur:
        buckets.append(Bucket(len(buckets), cur))
    return buckets


MB = 1 << 20


def cap_elems(cap_mb: float) -> int:
    return int(cap_mb * MB) // 4


# ----------------------------------------------------------------------------- model families
def resnet50_tensors(width: int = 64, blocks: Tuple[int, ...] = (3, 4, 6, 3), classes: int = 1000,
                     ) -> List[TensorSpec]:
    """ResNet-50 layout (bottleneck, expansion 4). Convs eligible; BN and the fc head FP32
    ('separates the convolutional backbone from the final classifier head')."""
    ts: List[TensorSpec] = []

    def conv(name, cout, cin, k):
        ts.append(TensorSpec(name + ".weight", cout * cin * k * k, True))

    def bn(name, c):
        ts.append(TensorSpec(name + ".weight", c, False))
        ts.append(TensorSpec(name + ".bias", c, False))

    conv("conv1", width, 3, 7)
    bn("bn1", width)
    cin = width
    for s, nb in enumerate(blocks):
        w = width * (2 ** s)
        for b in range(nb):
            p = f"layer{s + 1}.{b}"
            conv(p + ".conv1", w, cin, 1); bn(p + ".bn1", w)
            conv(p + ".conv2", w, w, 3); bn(p + ".bn2", w)
            conv(p + ".conv3", 4 * w, w, 1); bn(p + ".bn3", 4 * w)
            if b == 0:
                conv(p + ".downsample.0", 4 * w, cin, 1); bn(p + ".downsample.1", 4 * w)
            cin = 4 * w
    ts.append(TensorSpec("fc.weight", classes * cin, False))
    ts.append(TensorSpec("fc.bias", classes, False))
    return ts


def vit_tensors(d: int = 768, depth: int = 12, mlp: int = 3072, patch: int = 16, tokens: int = 197,
                classes: int = 1000) -> List[TensorSpec]:
    """ViT-B/16 layout. The 4 weight matrices of each block eligible; cls/pos/patch embeddings,
    LayerNorms, biases and head FP32."""
    ts = [TensorSpec("cls_token", d, False), TensorSpec("pos_embed", tokens * d, False),
          TensorSpec("patch_embed.proj.weight", d * 3 * patch * patch, False),
          TensorSpec("patch_embed.proj.bias", d, False)]
    for i in range(depth):
        p = f"blocks.{i}"
        ts += [TensorSpec(p + ".norm1.weight", d, False, i), TensorSpec(p + ".norm1.bias", d, False, i),
               TensorSpec(p + ".attn.qkv.weight", 3 * d * d, True, i),
               TensorSpec(p + ".attn.qkv.bias", 3 * d, False, i),
               TensorSpec(p + ".attn.proj.weight", d * d, True, i),
               TensorSpec(p + ".attn.proj.bias", d, False, i),
               TensorSpec(p + ".norm2.weight", d, False, i), TensorSpec(p + ".norm2.bias", d, False, i),
               TensorSpec(p + ".mlp.fc1.weight", mlp * d, True, i),
               TensorSpec(p + ".mlp.fc1.bias", mlp, False, i),
               TensorSpec(p + ".mlp.fc2.weight", d * mlp, True, i),
               TensorSpec(p + ".mlp.fc2.bias", d, False, i)]
    ts += [TensorSpec("norm.weight", d, False), TensorSpec("norm.bias", d, False),
           TensorSpec("head.weight", classes * d, False), TensorSpec("head.bias", classes, False)]
    return ts


def gpt2_tensors(d: int = 2048, layers: int = 24, mlp: int = 8192, vocab: int = 50257,
                 ctx: int = 1024) -> List[TensorSpec]:
    """GPT-2-1.3B-shaped layout (head tied to wte). Weight matrices eligible; embeddings,
    LayerNorms and biases FP32 (Table 4 L333-338 for the LM family)."""
    ts = [TensorSpec("wte", vocab * d, False), TensorSpec("wpe", ctx * d, False)]
    for i in range(layers):
        p = f"h.{i}"
        ts += [TensorSpec(p + ".ln_1.weight", d, False, i), TensorSpec(p + ".ln_1.bias", d, False, i),
               TensorSpec(p + ".attn.c_attn.weight", d * 3 * d, True, i),
               TensorSpec(p + ".attn.c_attn.bias", 3 * d, False, i),
               TensorSpec(p + ".attn.c_proj.weight", d * d, True, i),
               TensorSpec(p + ".attn.c_proj.bias", d, False, i),
               TensorSpec(p + ".ln_2.weight", d, False, i), TensorSpec(p + ".ln_2.bias", d, False, i),
               TensorSpec(p + ".mlp.c_fc.weight", d * mlp, True, i),
               TensorSpec(p + ".mlp.c_fc.bias", mlp, False, i),
               TensorSpec(p + ".mlp.c_proj.weight", mlp * d, True, i),
               TensorSpec(p + ".mlp.c_proj.bias", d, False, i)]
    ts += [TensorSpec("ln_f.weight", d, False), TensorSpec("ln_f.bias", d, False)]
    return ts


# ----------------------------------------------------------------------------- the five configs
TINY_LEN = [16384, 4096, 8192, 4096, 16384, 4096, 8192, 4096]
TINY_FP32 = (1, 3, 7)


def tiny() -> Config:
    ts = [TensorSpec(f"t{i}", l, i not in TINY_FP32) for i, l in enumerate(TINY_LEN)]
    # one bucket, tensors already in bucket order
    return Config("tiny", 0, 4, [Bucket(0, ts)], "gauss", 1e-4, 1e-1, "loguniform", 0.01)


def resnet50(small: bool = False) -> Config:
    if small:   # same structure, 1/8 width, 10 classes: ~0.4 M params, cap scaled alike
        ts, cap = resnet50_tensors(width=8, classes=10), cap_elems(25) // 64
    else:
        ts, cap = resnet50_tensors(), cap_elems(25)
    return Config("resnet50" + ("_small" if small else ""), 1, 8, bucketize(ts, cap), "gauss",
                  1e-5, 1e-2, "loguniform", 0.005)


def vit_b16(small: bool = False) -> Config:
    if small:
        ts, cap = vit_tensors(d=48, depth=3, mlp=192, patch=4, tokens=17, classes=10), cap_elems(25) // 256
    else:
        ts, cap = vit_tensors(), cap_elems(25)
    return Config("vit_b16" + ("_small" if small else ""), 2, 16, bucketize(ts, cap), "student3",
                  1e-5, 1e-2, "loguniform", 0.0)


def gpt2_1p3b(small: bool = False) -> Config:
    if small:
        ts, cap = gpt2_tensors(d=64, layers=3, mlp=256, vocab=1031, ctx=32), cap_elems(100) // 1024
        nan_bucket = 1
    else:
        ts, cap = gpt2_tensors(), cap_elems(100)
        nan_bucket = 1
    return Config("gpt2_1p3b" + ("_small" if small else ""), 3, 8, bucketize(ts, cap), "gauss",
                  5e-4, 1e-3, "gpt_layer", 0.0, nan_frac=0.001, nan_bucket=nan_bucket, nan_worker=3)


SWEEP_W = (2, 8, 32, 64, 128)


def sweep(W: int, n: int = 6_553_600) -> Config:
    ts = [TensorSpec("flat", n, True)]
    return Config(f"sweep_w{W}", 4, W, [Bucket(0, ts)], "gauss", 1e-3, 1e-3, "const", 0.0)


def paper_local_count(n: int) -> Config:
    """PAPER L456 context rows: 8 x 131K and 8 x 524K, all-eligible."""
    ts = [TensorSpec("flat", n, True)]
    return Config(f"local_count_8x{n // 1024}K", 5, 8, [Bucket(0, ts)], "gauss", 1e-3, 1e-3, "const", 0.0)


def get(name: str, small: bool = False) -> Config:
    if name == "tiny":
        return tiny()
    if name == "resnet50":
        return resnet50(small)
    if name == "vit_b16":
        return vit_b16(small)
    if name == "gpt2_1p3b":
        return gpt2_1p3b(small)
    if name.startswith("sweep_w"):
        return sweep(int(name[len("sweep_w"):]), 65_536 * 3 + 77 if small else 6_553_600)
    raise KeyError(name)
