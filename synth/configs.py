"""Model hyper-parameters and the five BASELINE.json workloads (shapes only)."""
from __future__ import annotations
from dataclasses import dataclass, field

BASE_SEED = 260117554          # arxiv id 2601.17554
N_FEAT = 55                    # BASELINE.json: 55 fp32 input features per element
N_TYPES = 4                    # track, ECAL, HCAL, HF (type id 1..4; 0 = pad row)
N_CLASSES = 9                  # BASELINE.json: 9-class logits
REG_DIMS = (1, 1, 2, 1)        # pT', eta, (sin phi, cos phi), E'  (reading A11)
N_REG = sum(REG_DIMS)          # 5 regressions


@dataclass(frozen=True)
class ModelCfg:
    n_layers: int
    d_model: int
    n_heads: int
    d_ff: int
    activation: str = "gelu"   # "gelu" (exact erf form) or "relu" (paper L156)
    final_ln: bool = True
    ln_eps: float = 1e-5
    n_feat: int = N_FEAT
    n_types: int = N_TYPES
    n_classes: int = N_CLASSES
    reg_dims: tuple = REG_DIMS
    # paper-faithful topology (Fig. 2): n_stacks = 2 runs two parallel encoders on the shared
    # embedding (stack 0 = classification, stack 1 = regression); binary_head adds the "valid" head on stack 0
    n_stacks: int = 1
    binary_head: bool = False

    @property
    def head_dim(self) -> int:
        return self.d_model // self.n_heads


# key -> (model, workload description).  Workload draws live in events.py.
CONFIGS = {
    "cfg1": ModelCfg(n_layers=2, d_model=64, n_heads=4, d_ff=256),
    "cfg2": ModelCfg(n_layers=3, d_model=256, n_heads=8, d_ff=1024),
    "cfg3": ModelCfg(n_layers=6, d_model=256, n_heads=8, d_ff=1024),
    "cfg4": ModelCfg(n_layers=6, d_model=512, n_heads=16, d_ff=2048),
    "cfg5a": ModelCfg(n_layers=8, d_model=512, n_heads=8, d_ff=2048),
    "cfg5b": ModelCfg(n_layers=8, d_model=512, n_heads=8, d_ff=2048),
    # paper-faithful block shape: d=256, 16 heads x 16, ReLU, 3 blocks
    "paper": ModelCfg(n_layers=3, d_model=256, n_heads=16, d_ff=1024, activation="relu"),
    # the paper's network (L156): two parallel 3-block encoders, d=256, 16 x 16, ReLU, six heads incl. binary
    "paper2": ModelCfg(n_layers=3, d_model=256, n_heads=16, d_ff=1024, activation="relu", n_stacks=2, binary_head=True),
}
CFG_INDEX = {"cfg1": 1, "cfg2": 2, "cfg3": 3, "cfg4": 4, "cfg5a": 5, "cfg5b": 6, "paper": 7, "paper2": 8}


def model_cfg(name: str) -> ModelCfg:
    return CONFIGS[name]


def stack_prefix(m: ModelCfg, s: int) -> str:
    """Name prefix of encoder stack s: "" for the single-stack configs, "enc<s>." for n_stacks = 2."""
    return "" if m.n_stacks == 1 else f"enc{s}."


def weight_names(m: ModelCfg):
    """Ordered (name, shape) list == the blob tensor order (include/mlpf.h)."""
    d, F, dff = m.d_model, m.n_feat, m.d_ff
    out = []
    for t in range(1, m.n_types + 1):
        out += [(f"emb.{t}.W1", (d, F)), (f"emb.{t}.b1", (d,)),
                (f"emb.{t}.W2", (d, d)), (f"emb.{t}.b2", (d,))]
    for s in range(m.n_stacks):
        for l in range(m.n_layers):
            p = f"{stack_prefix(m, s)}layer.{l}."
            out += [(p + "ln1.g", (d,)), (p + "ln1.b", (d,)),
                    (p + "Wqkv", (3 * d, d)), (p + "bqkv", (3 * d,)),
                    (p + "Wo", (d, d)), (p + "bo", (d,)),
                    (p + "ln2.g", (d,)), (p + "ln2.b", (d,)),
                    (p + "W1", (dff, d)), (p + "b1", (dff,)),
                    (p + "W2", (d, dff)), (p + "b2", (d,))]
    for s in range(m.n_stacks):
        out += [(f"{stack_prefix(m, s)}lnf.g", (d,)), (f"{stack_prefix(m, s)}lnf.b", (d,))]
    if m.binary_head:
        out += [("bin.W1", (d, d)), ("bin.b1", (d,)), ("bin.W2", (1, d)), ("bin.b2", (1,))]
    out += [("cls.W1", (d, d)), ("cls.b1", (d,)),
            ("cls.W2", (m.n_classes, d)), ("cls.b2", (m.n_classes,))]
    for k, rk in enumerate(m.reg_dims):
        out += [(f"reg.{k}.W1", (d, d)), (f"reg.{k}.b1", (d,)),
                (f"reg.{k}.W2", (rk, d)), (f"reg.{k}.b2", (rk,))]
    return out


def param_count(m: ModelCfg) -> int:
    n = 0
    for _, shp in weight_names(m):
        k = 1
        for s in shp:
            k *= s
        n += k
    return n
