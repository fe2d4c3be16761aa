"""The five BASELINE.json configs as plain data (shapes + scenario parameters).

Nothing here computes a partition, a plan or an address: widths that the method
derives by formula are left as ``None`` and each side (library / oracle) fills
them in with its own ``partition``.  Open points resolved as in DESIGN.md
("Readings"): failed rank for config 4, failure sequence for config 5, explicit
unequal OLD widths for configs 1 and 3.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

# granularity classes (PAPER.md:45 "attention and linear layers", :96 "head-groups")
HEAD, FFN, EXPERT, VOCAB = "head", "ffn", "expert", "vocab"
CLASSES = (HEAD, FFN, EXPERT, VOCAB)


@dataclass(frozen=True)
class ModelShape:
    name: str
    n_layers: int
    hidden: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    ffn: int = 0            # dense FFN width (0 for MoE-only layers)
    vocab: int = 0          # 0 => no embedding / lm_head in this config
    n_experts: int = 0
    expert_ffn: int = 0
    top_k: int = 0
    dtype: str = "bf16"     # "bf16" | "fp16"
    elem_bytes: int = 2
    init_std: float = 0.02

    @property
    def q_per_kv(self) -> int:
        return self.n_q_heads // self.n_kv_heads


@dataclass(frozen=True)
class KVShape:
    n_seqs: int
    seq_len: int
    block_size: int = 16
    pool_slack: float = 1.25   # pool blocks = ceil(slack * live blocks)


@dataclass(frozen=True)
class Scenario:
    n_old: int
    failed: Tuple[int, ...]                  # ranks that die, in order (one reshard each)
    old_policy: str = "floor"                # policy used where old widths are not explicit
    new_policy: str = "floor"
    old_widths: Dict[str, Tuple[int, ...]] = field(default_factory=dict)   # explicit unequal OLD widths


@dataclass(frozen=True)
class Config:
    index: int
    key: str
    model: ModelShape
    kv: KVShape
    scenario: Scenario
    tokens: int = 4      # batch for the shard-linear check
    note: str = ""


@dataclass(frozen=True)
class TensorSpec:
    """One sharded tensor: ``total_units`` units of ``unit_bytes`` contiguous bytes each.

    ``transposed`` marks row-parallel weights, stored ``[in][out]`` so that a unit
    interval is one contiguous byte interval (reading L1).
    ``features_per_unit`` = rows of the stored 2-D matrix per unit; ``row_elems`` =
    elements per stored row.
    """
    name: str
    klass: str
    layer: int            # -1 for model-level tensors
    total_units: int
    unit_bytes: int
    features_per_unit: int
    row_elems: int
    transposed: bool
    stream: int           # generator stream id (unique per tensor)


def tensor_inventory(cfg: Config) -> List[TensorSpec]:
    m = cfg.model
    eb = m.elem_bytes
    out: List[TensorSpec] = []
    sid = 0

    def add(name, klass, layer, units, fpu, row_elems, transposed):
        nonlocal sid
        out.append(TensorSpec(name, klass, layer, units, fpu * row_elems * eb, fpu, row_elems, transposed, sid))
        sid += 1

    g = m.q_per_kv * m.head_dim      # Q rows per KV-head group
    for l in range(m.n_layers):
        add(f"l{l}.wq", HEAD, l, m.n_kv_heads, g, m.hidden, False)
        add(f"l{l}.wk", HEAD, l, m.n_kv_heads, m.head_dim, m.hidden, False)
        add(f"l{l}.wv", HEAD, l, m.n_kv_heads, m.head_dim, m.hidden, False)
        add(f"l{l}.wo_t", HEAD, l, m.n_kv_heads, g, m.hidden, True)
        if m.ffn:
            add(f"l{l}.gate", FFN, l, m.ffn, 1, m.hidden, False)
            add(f"l{l}.up", FFN, l, m.ffn, 1, m.hidden, False)
            add(f"l{l}.down_t", FFN, l, m.ffn, 1, m.hidden, True)
        if m.n_experts:
            # one unit = one whole expert matrix (north_star: "expert granularity")
            add(f"l{l}.exp_gate", EXPERT, l, m.n_experts, m.expert_ffn, m.hidden, False)
            add(f"l{l}.exp_up", EXPERT, l, m.n_experts, m.expert_ffn, m.hidden, False)
            add(f"l{l}.exp_down_t", EXPERT, l, m.n_experts, m.expert_ffn, m.hidden, True)
    if m.vocab:
        add("embed", VOCAB, -1, m.vocab, 1, m.hidden, False)
        add("lm_head", VOCAB, -1, m.vocab, 1, m.hidden, False)
    return out


def class_units(cfg: Config) -> Dict[str, int]:
    m = cfg.model
    d = {HEAD: m.n_kv_heads}
    if m.ffn:
        d[FFN] = m.ffn
    if m.n_experts:
        d[EXPERT] = m.n_experts
    if m.vocab:
        d[VOCAB] = m.vocab
    return d


_TINY = ModelShape("tiny-dense", 1, 256, 8, 4, 32, ffn=688, dtype="fp16")
_QWEN14 = ModelShape("qwen3-14b-shape", 40, 5120, 40, 8, 128, ffn=17408, vocab=151936)
_LLAMA8 = ModelShape("llama3-8b-shape", 32, 4096, 32, 8, 128, ffn=14336, vocab=128256)
_QWEN30A3 = ModelShape("qwen3-30b-a3b-shape-24l", 24, 2048, 32, 4, 128,
                       n_experts=128, expert_ffn=768, top_k=8)

CONFIGS: Dict[str, Config] = {
    "1": Config(1, "1", _TINY, KVShape(2, 128), Scenario(
        4, (2,), old_widths={HEAD: (1, 1, 1, 1), FFN: (160, 176, 184, 168)}),
        tokens=4, note="tiny dense layer, CPU-seconds scale"),
    "2": Config(2, "2", _QWEN14, KVShape(64, 2048), Scenario(
        4, (1,), new_policy="ceil_first"),
        note="headline: Qwen3-14B shape 4->3, KV heads 3/3/2 (BASELINE.json)"),
    "2b": Config(2, "2b", _QWEN14, KVShape(64, 2048), Scenario(4, (1,)),
                 note="same, the paper's floor-boundary policy (heads 2/3/3)"),
    "3": Config(3, "3", _LLAMA8, KVShape(128, 1024), Scenario(
        8, (5,), old_widths={FFN: (1856, 1728, 1920, 1664, 1824, 1760, 1888, 1696)}),
        note="Llama-3-8B shape 8->7, explicit unequal OLD FFN widths"),
    "4": Config(4, "4", _QWEN30A3, KVShape(32, 4096), Scenario(4, (1,)),
                note="Qwen3-30B-A3B shape (24 layers) 4->3, expert granularity"),
    "5a": Config(5, "5a", _LLAMA8, KVShape(128, 1024), Scenario(8, (5, 0, 7)),
                 note="sequential failures 8->7->6->5"),
}


def get_config(key) -> Config:
    return CONFIGS[str(key)]


# config 5b: copy-kernel microbenchmark recipe (n intervals, log-uniform sizes).
# The stated 256 B - 64 MB range cannot hold for large n; the upper bound is clipped
# so that the total stays <= 32 GiB (R-5b).
MICROBENCH_HI = {100: 64 << 20, 1000: 64 << 20, 10_000: 32 << 20, 100_000: 2 << 20, 1_000_000: 128 << 10}
MICROBENCH_LO = 256


def scaled(cfg: Config, n_layers: Optional[int] = None, n_seqs: Optional[int] = None,
           seq_len: Optional[int] = None, vocab: Optional[int] = None) -> Config:
    """Same shape with fewer layers / sequences / no embedding (bounded samples of a workload)."""
    import dataclasses
    m = cfg.model if n_layers is None else dataclasses.replace(cfg.model, n_layers=n_layers)
    if vocab is not None:
        m = dataclasses.replace(m, vocab=vocab)
    kv = cfg.kv
    if n_seqs is not None or seq_len is not None:
        kv = dataclasses.replace(kv, n_seqs=n_seqs or kv.n_seqs, seq_len=seq_len or kv.seq_len)
    return dataclasses.replace(cfg, model=m, kv=kv)
