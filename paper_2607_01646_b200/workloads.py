"""Synthetic workloads: shard shapes and seeded input generators.

This module holds NONE of the method's arithmetic (no AdamW, no rounding, no
partitioning of the flat space, no header packing).  It only
  * lists, for each BASELINE.json config, the tensors a rank holds after TP/PP
    slicing (architecture arithmetic), and
  * draws seeded parameter / gradient values with the distributions the configs
    name (BASELINE.json:configs[0..4]).
Both the oracle-side tests and the CUDA-side tests/bench take their inputs from
here: values are generated ONCE (on whichever device) and the same bits are
handed to both sides; they are never regenerated independently.

The paper trains real GPT models on real data; none of that
is available here, so these inputs stand in for it.  Only sizes, segment
boundaries and value distributions matter to this path.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Sequence, Tuple

import torch

# ----------------------------------------------------------------------------
# tensor lists
# ----------------------------------------------------------------------------


@dataclass(frozen=True)
class TensorSpec:
    name: str
    numel: int
    group: int  # gradient-scale group (layer index; -1.. for embeddings etc.)


def gpt_tensors(layers: int, hidden: int, vocab: int, seq: int) -> List[TensorSpec]:
    """GPT-2/3 style decoder with biases, LayerNorm and a tied embedding.

    Per layer 12h^2 + 13h; total V*h + S*h + L*per + 2h.
    """
    h = hidden
    t: List[TensorSpec] = [
        TensorSpec("word_embeddings.weight", vocab * h, 0),
        TensorSpec("position_embeddings.weight", seq * h, 0),
    ]
    for l in range(layers):
        g = l + 1
        pre = f"layers.{l}."
        t += [
            TensorSpec(pre + "ln1.weight", h, g),
            TensorSpec(pre + "ln1.bias", h, g),
            TensorSpec(pre + "attn.qkv.weight", 3 * h * h, g),
            TensorSpec(pre + "attn.qkv.bias", 3 * h, g),
            TensorSpec(pre + "attn.proj.weight", h * h, g),
            TensorSpec(pre + "attn.proj.bias", h, g),
            TensorSpec(pre + "ln2.weight", h, g),
            TensorSpec(pre + "ln2.bias", h, g),
            TensorSpec(pre + "mlp.fc1.weight", 4 * h * h, g),
            TensorSpec(pre + "mlp.fc1.bias", 4 * h, g),
            TensorSpec(pre + "mlp.fc2.weight", 4 * h * h, g),
            TensorSpec(pre + "mlp.fc2.bias", h, g),
        ]
    t += [
        TensorSpec("final_ln.weight", h, layers + 1),
        TensorSpec("final_ln.bias", h, layers + 1),
    ]
    return t


def llama_tensors(
    layers: int,
    hidden: int,
    ffn: int,
    vocab: int,
    tp_size: int = 1,
    pp_size: int = 1,
    tp_rank: int = 0,
    pp_rank: int = 0,
) -> List[TensorSpec]:
    """LLaMA style decoder (no biases, RMSNorm, untied head), after TP/PP slicing.

    TP splits every matrix 1/tp (norms replicated); PP gives each stage
    layers/pp consecutive layers, the embedding to the first stage and the final
    norm + head to the last.  Per layer 4h^2 + 3*h*ffn + 2h.
    """
    h = hidden
    assert layers % pp_size == 0 and (h * h) % tp_size == 0 and (h * ffn) % tp_size == 0
    assert 0 <= tp_rank < tp_size and 0 <= pp_rank < pp_size
    t: List[TensorSpec] = []
    if pp_rank == 0:
        t.append(TensorSpec("tok_embeddings.weight", vocab * h // tp_size, 0))
    per = layers // pp_size
    for l in range(pp_rank * per, (pp_rank + 1) * per):
        g = l + 1
        pre = f"layers.{l}."
        t += [
            TensorSpec(pre + "attention_norm.weight", h, g),
            TensorSpec(pre + "attention.wq.weight", h * h // tp_size, g),
            TensorSpec(pre + "attention.wk.weight", h * h // tp_size, g),
            TensorSpec(pre + "attention.wv.weight", h * h // tp_size, g),
            TensorSpec(pre + "attention.wo.weight", h * h // tp_size, g),
            TensorSpec(pre + "ffn_norm.weight", h, g),
            TensorSpec(pre + "feed_forward.w1.weight", h * ffn // tp_size, g),
            TensorSpec(pre + "feed_forward.w3.weight", h * ffn // tp_size, g),
            TensorSpec(pre + "feed_forward.w2.weight", h * ffn // tp_size, g),
        ]
    if pp_rank == pp_size - 1:
        t += [
            TensorSpec("norm.weight", h, layers + 1),
            TensorSpec("output.weight", vocab * h // tp_size, layers + 1),
        ]
    return t


# ----------------------------------------------------------------------------
# configs (BASELINE.json:configs[0..4])
# ----------------------------------------------------------------------------


@dataclass(frozen=True)
class Hyper:
    lr: float = 3e-4
    beta1: float = 0.9
    beta2: float = 0.95
    eps: float = 1e-8
    wd: float = 0.1
    max_grad_norm: float = 0.0  # <= 0: no clip


@dataclass(frozen=True)
class Workload:
    key: str
    title: str
    tensors: Tuple[TensorSpec, ...]
    dp_size: int
    dp_rank: int = 0
    tp_size: int = 1
    tp_rank: int = 0
    pp_size: int = 1
    pp_rank: int = 0
    hyper: Hyper = field(default_factory=Hyper)
    grad_kind: str = "normal"  # "normal" | "heavy_tail"
    scale_per: str = "group"   # "tensor" | "group" : granularity of the U[0.5,2] scale
    n_expected: int = 0        # per-rank fp32 elements the config text / Appendix C states
    seed: int = 0
    decay_groups: bool = False  # biases and norm weights are flagged no-decay
    precision: str = "bf16"     # "bf16": bf16 grads + bf16 copy (north_star); "fp32": the paper's
    no_decay_ids: Tuple[int, ...] = ()  # extra tensor indices flagged no-decay (ad-hoc test workloads)

    @property
    def total_numel(self) -> int:
        return sum(t.numel for t in self.tensors)

    def layout(self) -> List[Tuple[int, int]]:
        """[(numel, tensor_id)] in list order — the argument of phx_shard_create / the oracle's a0."""
        return [(t.numel, i) for i, t in enumerate(self.tensors)]

    def flags(self) -> List[int]:
        """Per-tensor flags for phx_tensor_desc_t.flags / the oracle's a0: bit 0 (no decay) on biases
        and normalisation weights when decay_groups is on (the usual AdamW parameter groups)."""
        nd = ("bias", "ln1.", "ln2.", "final_ln.", "norm.") if self.decay_groups else ()
        return [1 if (i in self.no_decay_ids or any(k in t.name for k in nd)) else 0
                for i, t in enumerate(self.tensors)]


def _mk() -> dict:
    w = {}
    w["c1"] = Workload(
        "c1", "Tiny GPT shard: 4L h256 4 heads V8192 S128, dp4 rank0",
        tuple(gpt_tensors(4, 256, 8192, 128)), dp_size=4, scale_per="tensor",
        n_expected=1_322_368)
    w["c2"] = Workload(
        "c2", "GPT-3 1.3B-style shard: 24L h2048 V50304 S2048, dp8 rank0",
        tuple(gpt_tensors(24, 2048, 50304, 2048)), dp_size=8,
        n_expected=164_477_440)
    w["c3"] = Workload(
        "c3", "LLaMA-7B-style shard: 32L h4096 ffn11008 V32000, TP1 PP1 dp16 rank0, clip 1.0",
        tuple(llama_tensors(32, 4096, 11008, 32000)), dp_size=16,
        hyper=Hyper(max_grad_norm=1.0), grad_kind="heavy_tail",
        n_expected=421_150_976)
    t13 = tuple(llama_tensors(40, 5120, 13824, 32000, tp_size=2, pp_size=2))
    w["c4a"] = Workload(
        "c4a", "LLaMA-13B-style hot-swap shard (~200M as the config states): TP2 PP2, dp16 rank0",
        t13, dp_size=16, tp_size=2, pp_size=2, n_expected=203_379_200)
    w["c4b"] = Workload(
        "c4b", "LLaMA-13B-style hot-swap shard (architecture-derived): TP2 PP2, dp8 rank0",
        t13, dp_size=8, tp_size=2, pp_size=2, n_expected=406_758_400)
    w["c5"] = Workload(
        "c5", "LLaMA-65B-style shard: 80L h8192 ffn22016, TP8 PP8, dp4 rank0 ((tp0,pp0) slice)",
        tuple(llama_tensors(80, 8192, 22016, 32000, tp_size=8, pp_size=8)),
        dp_size=4, tp_size=8, pp_size=8, n_expected=261_201_920)
    return w


CONFIGS = _mk()


def tiny_workload(numels: Sequence[int], dp_size: int, dp_rank: int = 0, **kw) -> Workload:
    """Ad-hoc small workload for tests (ragged tensor sizes, several ranks...)."""
    ts = tuple(TensorSpec(f"t{i}", int(n), i) for i, n in enumerate(numels))
    return Workload("tiny", "ad-hoc test workload", ts, dp_size=dp_size, dp_rank=dp_rank, **kw)


# ----------------------------------------------------------------------------
# seeded generators.  `segments` = [(tensor_id, off_in_shard, length)] comes from
# whoever partitioned the shard (the oracle's a0 in oracle-side tests, the
# library's phx_shard_segments on the CUDA side) — not computed here.
# ----------------------------------------------------------------------------

Segment = Tuple[int, int, int]  # tensor_id, offset in shard, length


def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed) & 0x7FFFFFFFFFFFFFFF)
    return g


def init_params(n: int, n_padded: int, seed: int = 0, device="cpu") -> torch.Tensor:
    """fp32 master params ~ N(0, 0.02) (GPT init std); pad lanes [n, n_padded) are zero."""
    p = torch.zeros(n_padded, dtype=torch.float32, device=device)
    if n > 0:
        p[:n].normal_(0.0, 0.02, generator=_gen(seed * 1_000_003 + 17, device))
    return p


def group_scales(wl: Workload, seed: int = 0) -> List[float]:
    """One U[0.5, 2] scale per tensor (indexed by tensor_id), shared inside a layer
    when wl.scale_per == 'group'.  Drawn once, on the CPU generator, from `seed`."""
    g = _gen(seed * 7_919 + 101, "cpu")
    if wl.scale_per == "tensor":
        u = torch.rand(len(wl.tensors), generator=g, dtype=torch.float64)
        return [0.5 + 1.5 * float(x) for x in u]
    ngroups = max(t.group for t in wl.tensors) + 1
    u = torch.rand(ngroups, generator=g, dtype=torch.float64)
    return [0.5 + 1.5 * float(u[t.group]) for t in wl.tensors]


def gen_grads(
    wl: Workload,
    segments: Sequence[Segment],
    n_padded: int,
    step: int,
    seed: int = 0,
    device="cpu",
    chunk: int = 1 << 26,
    dtype: torch.dtype = torch.bfloat16,
) -> torch.Tensor:
    """Gradients for one step, already reduce-scattered to this rank's shard: bf16 (default) or
    float32 (`dtype`, the paper's all-FP32 setting, PAPER.md:270 — the same draws, not cast down).

    'normal'     : N(0, 1e-3) times the tensor's U[0.5,2] scale.
    'heavy_tail' : the same, except a Bernoulli(0.01) subset is 1e-3 * Student-t(df=3)
                   times the scale.
    Cast to bf16 with torch's round-to-nearest-even; pad lanes are zero.  The
    returned BITS are the input of record for both sides.
    """
    scales = group_scales(wl, seed)
    gen = _gen(seed * 2_654_435_761 + 1_000_000_007 * (step + 1), device)
    out = torch.zeros(n_padded, dtype=dtype, device=device)
    for tid, off, length in segments:
        s = 1e-3 * scales[tid]
        for c0 in range(0, length, chunk):
            c = min(chunk, length - c0)
            z = torch.randn(c, generator=gen, dtype=torch.float32, device=device)
            if wl.grad_kind == "heavy_tail":
                mask = torch.rand(c, generator=gen, dtype=torch.float32, device=device) < 0.01
                k = int(mask.sum().item())
                if k:
                    num = torch.randn(k, generator=gen, dtype=torch.float32, device=device)
                    chi = torch.randn(3, k, generator=gen, dtype=torch.float32, device=device)
                    den = torch.sqrt((chi * chi).sum(0) / 3.0)
                    z[mask] = num / den
            out[off + c0: off + c0 + c] = (z * s).to(dtype)
    return out
