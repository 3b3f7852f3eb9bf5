"""Seeded synthetic U(1)-labelled block-sparse operator sets and MPS site tensors.

Stand-in for the FeMoco CAS(54,54) / CAS(113,76) scratch data of PAPER.md §IV (L148, L158,
L186): those integrals, MPS states and the authors' code are not available; these sets take
their *shape* — bond dimension D up to the U(1) ~15400 of L192, many operators sharing one
block structure (Fig 4(a), L75), 4 local states per site tensor (Eq. 2), non-zero sectors
selected by quantum-number conservation (L63).  Recipe: SURVEY.md §8(d), restated in DESIGN.md.

Only *inputs* are built here (labels, extents, tensor records, where each dense block lives in
the source pool).  Stream sizes, padding and offsets are the serializer's business and are not
computed in this module.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 241204676

# descriptor record of one tensor, 32 bytes (include/bs.h bs_tensor_rec)
TENSOR_REC_DTYPE = np.dtype(
    [("rank", "<u4"), ("first_block", "<u4"), ("n_blocks", "<u4"), ("dq", "<i4", (2,)),
     ("sign", "i1", (4,)), ("tag", "<u4"), ("reserved", "<u4")]
)
assert TENSOR_REC_DTYPE.itemsize == 32

# local (N, 2Sz) labels of one spinful orbital: |0>, |up>, |dn>, |updn>
LOCAL_LABELS = np.array([(0, 0), (1, 1), (1, -1), (2, 0)], dtype=np.int32)


def selection_rules() -> np.ndarray:
    """The 13 parity-consistent (dN, d2Sz) rules with dN in {0,+-1,+-2}, dSz in {0,+-1/2,+-1}."""
    return np.array(
        [(0, 0), (1, 1), (1, -1), (-1, 1), (-1, -1), (2, 0), (-2, 0),
         (2, 2), (2, -2), (-2, 2), (-2, -2), (0, 2), (0, -2)], dtype=np.int32)


def label_grid(S: int, M: int, N0: int) -> np.ndarray:
    """First S labels (N, m) enumerated N = N0, N0+1, ...; m = -M_N .. +M_N step 2, m == N (mod 2)."""
    out = []
    N = N0
    while len(out) < S:
        MN = M if (M - N) % 2 == 0 else M - 1
        for m in range(-MN, MN + 1, 2):
            out.append((N, m))
            if len(out) == S:
                break
        N += 1
    return np.array(out, dtype=np.int32)


def dims_multinomial(rng: np.random.Generator, D: int, S: int) -> np.ndarray:
    return (1 + rng.multinomial(D - S, np.full(S, 1.0 / S))).astype(np.uint32)


def dims_lognormal(rng: np.random.Generator, D: int, S: int, sigma: float) -> np.ndarray:
    w = np.exp(sigma * rng.standard_normal(S))
    x = (D - S) * w / w.sum()
    fl = np.floor(x)
    d = 1 + fl.astype(np.int64)
    rem = int(D - d.sum())
    if rem > 0:
        order = np.argsort(-(x - fl), kind="stable")
        d[order[:rem]] += 1
    assert d.sum() == D and d.min() >= 1
    return d.astype(np.uint32)


def _label_index(labels: np.ndarray) -> dict:
    return {(int(n), int(m)): i for i, (n, m) in enumerate(labels)}


def _operator_class(labels, dims, rule):
    """Blocks (l -> r) with label_r = label_l + rule, in ascending l.  rank-2 record arrays."""
    idx = _label_index(labels)
    l_list, r_list = [], []
    for l, (n, m) in enumerate(labels):
        r = idx.get((int(n) + int(rule[0]), int(m) + int(rule[1])))
        if r is not None:
            l_list.append(l)
            r_list.append(r)
    l_arr = np.array(l_list, dtype=np.int64)
    r_arr = np.array(r_list, dtype=np.int64)
    nb = len(l_arr)
    qn = np.zeros((nb, 3, 2), dtype=np.int32)
    dim = np.ones((nb, 3), dtype=np.uint32)
    if nb:
        qn[:, 0, :] = labels[l_arr]
        qn[:, 1, :] = labels[r_arr]
        dim[:, 0] = dims[l_arr]
        dim[:, 1] = dims[r_arr]
    return qn, dim


def _site_class(labels, dims_l, dims_r):
    """Blocks (l, sigma, r) with label_l + q_sigma = label_r, ascending (l, sigma); shape (d_l, 1, d_r)."""
    idx = _label_index(labels)
    rows = []
    for l, (n, m) in enumerate(labels):
        for s, (qn_, qm_) in enumerate(LOCAL_LABELS):
            r = idx.get((int(n) + int(qn_), int(m) + int(qm_)))
            if r is not None:
                rows.append((l, s, r))
    nb = len(rows)
    qn = np.zeros((nb, 3, 2), dtype=np.int32)
    dim = np.ones((nb, 3), dtype=np.uint32)
    if nb:
        rows = np.array(rows, dtype=np.int64)
        qn[:, 0, :] = labels[rows[:, 0]]
        qn[:, 1, :] = LOCAL_LABELS[rows[:, 1]]
        qn[:, 2, :] = labels[rows[:, 2]]
        dim[:, 0] = dims_l[rows[:, 0]]
        dim[:, 2] = dims_r[rows[:, 2]]
    return qn, dim


@dataclass
class BlockSparseSet:
    """One scratch set: T tensors, B dense fp64 blocks, plus where each block lives in the source pool."""
    name: str
    seed: int
    tensors: np.ndarray            # [T] TENSOR_REC_DTYPE
    qn: np.ndarray                 # [B,3,2] int32, unused legs 0
    dim: np.ndarray                # [B,3]   uint32, unused legs 1
    pool_off: np.ndarray           # [B] uint64 byte offset of block i in the source pool (512-aligned)
    pool_bytes: int
    meta: dict = field(default_factory=dict)

    @property
    def n_tensors(self) -> int:
        return int(len(self.tensors))

    @property
    def n_blocks(self) -> int:
        return int(self.dim.shape[0])

    @property
    def legs(self) -> int:
        """Legs per block record: 3 (matrices and MPS site tensors), 4 for sets that hold order-4 tensors."""
        return int(self.dim.shape[1])

    @property
    def nelems(self) -> np.ndarray:
        d = self.dim.astype(np.uint64)
        n = d[:, 0].copy()
        for k in range(1, d.shape[1]):
            n = n * d[:, k]
        return n

    @property
    def data_bytes(self) -> int:
        return int(self.nelems.sum()) * 8


def _place(rng: np.random.Generator, nelems: np.ndarray, align: int, scatter: bool):
    """Pool offsets: blocks laid out in a seeded random permutation, each at an ``align``-byte boundary."""
    B = len(nelems)
    sz = (nelems.astype(np.int64) * 8 + (align - 1)) // align * align
    order = rng.permutation(B) if scatter else np.arange(B)
    off_sorted = np.zeros(B, dtype=np.int64)
    if B > 1:
        np.cumsum(sz[order][:-1], out=off_sorted[1:])
    pool_off = np.empty(B, dtype=np.uint64)
    pool_off[order] = off_sorted.astype(np.uint64)
    return pool_off, int(sz.sum())


def make_set(name: str, seed: int, D: int, S: int, M: int, N0: int, n_ops: int, n_site: int,
             dims: str, sigma: float = 0.0, rules: np.ndarray | None = None,
             pool_align: int = 512, scatter: bool = True) -> BlockSparseSet:
    rng = np.random.default_rng(seed)
    labels = label_grid(S, M, N0)
    draw = (lambda: dims_multinomial(rng, D, S)) if dims == "multinomial" \
        else (lambda: dims_lognormal(rng, D, S, sigma))
    bond = draw()
    if rules is None:
        rules = selection_rules()
    # structure classes: one per rule (shared by all operators of that rule: the "layers" of Fig 4(a)),
    # one per site tensor (left/right dims drawn independently)
    cls_qn, cls_dim = [], []
    for r in rules:
        q, d = _operator_class(labels, bond, r)
        cls_qn.append(q)
        cls_dim.append(d)
    for _ in range(n_site):
        dl, dr = draw(), draw()
        q, d = _site_class(labels, dl, dr)
        cls_qn.append(q)
        cls_dim.append(d)
    cls_nb = np.array([len(q) for q in cls_qn], dtype=np.int64)
    cls_start = np.concatenate([[0], np.cumsum(cls_nb)])[:-1]
    all_qn = np.concatenate(cls_qn) if cls_qn else np.zeros((0, 3, 2), np.int32)
    all_dim = np.concatenate(cls_dim) if cls_dim else np.ones((0, 3), np.uint32)

    T = n_ops + n_site
    cls_of = np.concatenate([np.arange(n_ops, dtype=np.int64) % len(rules),
                             len(rules) + np.arange(n_site, dtype=np.int64)])
    nb = cls_nb[cls_of] if T else np.zeros(0, np.int64)
    first = np.concatenate([[0], np.cumsum(nb)])[:-1] if T else np.zeros(0, np.int64)
    B = int(nb.sum())
    tensors = np.zeros(T, dtype=TENSOR_REC_DTYPE)
    tensors["rank"][:n_ops] = 2
    tensors["rank"][n_ops:] = 3
    tensors["first_block"] = first
    tensors["n_blocks"] = nb
    if n_ops:
        tensors["dq"][:n_ops] = rules[cls_of[:n_ops]]
        tensors["sign"][:n_ops] = (-1, 1, 0, 0)
    if n_site:
        tensors["dq"][n_ops:] = (0, 0)
        tensors["sign"][n_ops:] = (1, 1, -1, 0)
    tensors["tag"] = np.arange(T)

    t_of_b = np.repeat(np.arange(T, dtype=np.int64), nb)
    within = np.arange(B, dtype=np.int64) - first[t_of_b]
    src = cls_start[cls_of[t_of_b]] + within
    qn = np.ascontiguousarray(all_qn[src])
    dim = np.ascontiguousarray(all_dim[src])
    d64 = dim.astype(np.uint64)
    nelems = d64[:, 0] * d64[:, 1] * d64[:, 2]
    pool_off, pool_bytes = _place(rng, nelems, pool_align, scatter)
    meta = dict(D=D, S=S, M=M, N0=N0, n_ops=n_ops, n_site=n_site, dims=dims, sigma=sigma,
                pool_align=pool_align, scatter=scatter, bond_dims=bond,
                # the structure classes the tensors were drawn from (layered_view)
                cls_of=cls_of, cls_start=cls_start, cls_nb=cls_nb, cls_qn=all_qn, cls_dim=all_dim, n_rules=len(rules),
                rules=rules)
    return BlockSparseSet(name, seed, tensors, qn, dim, pool_off, pool_bytes, meta)


# descriptor records of the structure-shared ("layered") form of a set (include/bs.h bs_struct_rec, bs_layer_rec):
# the layers of PAPER Fig 4(a) (L75) name a structure; a structure owns one table of labelled sectors
STRUCT_REC_DTYPE = np.dtype([("rank", "<u4"), ("first_block", "<u4"), ("n_blocks", "<u4"), ("dq", "<i4", (2,)),
                             ("sign", "i1", (4,)), ("layer_bytes", "<u8")])
LAYER_REC_DTYPE = np.dtype([("structure", "<u4"), ("tag", "<u4"), ("offset", "<u8")])
assert STRUCT_REC_DTYPE.itemsize == 32 and LAYER_REC_DTYPE.itemsize == 16


def layered_view(bset: BlockSparseSet, keep_unused: bool = False) -> dict:
    """The same set in structure-shared form: operators drawn from one selection rule are LAYERS of one
    structure (Fig 4(a), L75); every site tensor is the single layer of its own structure.  Inputs only:
    ``layer_bytes`` / ``offset`` (the serializer's outputs) are left 0.  Block i of ``bset`` is entry i of the
    layered form's address list (layer-major, structure order inside a layer), so pools and addresses are shared.
    keep_unused: keep structures no layer refers to (n_ops < number of rules) instead of dropping them."""
    m = bset.meta
    cls_of, cls_start, cls_nb = m["cls_of"], m["cls_start"], m["cls_nb"]
    n_cls = len(cls_nb)
    used = np.zeros(n_cls, dtype=bool)
    used[cls_of] = True
    keep = np.ones(n_cls, dtype=bool) if keep_unused else used
    new_id = np.cumsum(keep) - 1
    ids = np.nonzero(keep)[0]
    structs = np.zeros(len(ids), dtype=STRUCT_REC_DTYPE)
    nb = cls_nb[ids]
    structs["n_blocks"] = nb
    structs["first_block"] = np.concatenate([[0], np.cumsum(nb)])[:-1] if len(ids) else np.zeros(0)
    is_op = ids < m["n_rules"]
    structs["rank"] = np.where(is_op, 2, 3)
    for k, c in enumerate(ids):
        if c < m["n_rules"]:
            structs["dq"][k] = m["rules"][c]
            structs["sign"][k] = (-1, 1, 0, 0)
        else:
            structs["dq"][k] = (0, 0)
            structs["sign"][k] = (1, 1, -1, 0)
    src = np.concatenate([np.arange(cls_start[c], cls_start[c] + cls_nb[c]) for c in ids]).astype(np.int64) \
        if len(ids) else np.zeros(0, np.int64)
    layers = np.zeros(bset.n_tensors, dtype=LAYER_REC_DTYPE)
    layers["structure"] = new_id[cls_of]
    layers["tag"] = bset.tensors["tag"]
    return dict(structs=structs, layers=layers, qn=np.ascontiguousarray(m["cls_qn"][src]),
                dim=np.ascontiguousarray(m["cls_dim"][src]))


def make_tree_set(name: str, seed: int, D: int = 24, S: int = 6, M: int = 2, n_nodes: int = 3, n_ops: int = 4,
                  pool_align: int = 512, scatter: bool = True) -> BlockSparseSet:
    """Order-4 tensors: the nodes of a tree tensor network state ("tree-like tensor network state methods";
    SURVEY §8(f) NEXT-4 "rank-4 tensors") — two child legs, a physical leg and a parent leg, U(1)-blocked like the order-3 MPS
    tensors of Eq. 2 (L47): block (a, b, sigma, c) kept iff label_a + label_b + q_sigma = label_c, shape (d_a, d_b, 1, d_c),
    sign (+1,+1,+1,-1), dq = 0.  Child-leg labels come from the grid G(S, M, 0), the parent leg from a grid wide enough to
    hold their sums; sector dims are multinomial draws summing to D per leg.  n_ops rank-2 operators on the child bond follow
    (selection rules as in make_set), so one set mixes ranks: their legs 3 and 4 are unused (dim 1, labels 0).
    Arrays have FOUR legs per block: qn [B][4][2], dim [B][4].  Inputs only (no stream arithmetic)."""
    rng = np.random.default_rng(seed)
    child = label_grid(S, M, 0)
    parent = label_grid(4 * S + 8, 2 * M + 2, 0)
    pidx = _label_index(parent)
    rules = selection_rules()
    qn_list, dim_list, recs = [], [], []
    first = 0
    for node in range(n_nodes):
        da, db = dims_multinomial(rng, D, S), dims_multinomial(rng, D, S)
        dc = dims_multinomial(rng, 2 * D, len(parent))
        rows = []
        for a, (na, ma) in enumerate(child):
            for b, (nb, mb) in enumerate(child):
                for sg, (ns, ms) in enumerate(LOCAL_LABELS):
                    c = pidx.get((int(na) + int(nb) + int(ns), int(ma) + int(mb) + int(ms)))
                    if c is not None:
                        rows.append((a, b, sg, c))
        rows = np.array(rows, dtype=np.int64).reshape(-1, 4)
        q = np.zeros((len(rows), 4, 2), np.int32)
        d = np.ones((len(rows), 4), np.uint32)
        if len(rows):
            q[:, 0], q[:, 1], q[:, 2], q[:, 3] = child[rows[:, 0]], child[rows[:, 1]], LOCAL_LABELS[rows[:, 2]], parent[rows[:, 3]]
            d[:, 0], d[:, 1], d[:, 3] = da[rows[:, 0]], db[rows[:, 1]], dc[rows[:, 3]]
        qn_list.append(q)
        dim_list.append(d)
        recs.append((4, first, len(rows), (0, 0), (1, 1, 1, -1), node, 0))
        first += len(rows)
    bond = dims_multinomial(rng, D, S)
    for k in range(n_ops):
        q3, d3 = _operator_class(child, bond, rules[k % len(rules)])
        q = np.zeros((len(q3), 4, 2), np.int32)
        d = np.ones((len(q3), 4), np.uint32)
        q[:, :3], d[:, :3] = q3, d3
        qn_list.append(q)
        dim_list.append(d)
        recs.append((2, first, len(q3), tuple(int(x) for x in rules[k % len(rules)]), (-1, 1, 0, 0), n_nodes + k, 0))
        first += len(q3)
    tensors = np.zeros(len(recs), dtype=TENSOR_REC_DTYPE)
    for i, r in enumerate(recs):
        tensors[i] = r
    qn = np.ascontiguousarray(np.concatenate(qn_list)) if qn_list else np.zeros((0, 4, 2), np.int32)
    dim = np.ascontiguousarray(np.concatenate(dim_list)) if dim_list else np.ones((0, 4), np.uint32)
    d64 = dim.astype(np.uint64)
    nelems = d64[:, 0] * d64[:, 1] * d64[:, 2] * d64[:, 3]
    pool_off, pool_bytes = _place(rng, nelems, pool_align, scatter)
    meta = dict(D=D, S=S, M=M, n_nodes=n_nodes, n_ops=n_ops, dims="multinomial", sigma=0.0, pool_align=pool_align, scatter=scatter)
    return BlockSparseSet(name, seed, tensors, qn, dim, pool_off, pool_bytes, meta)


# BASELINE.json configs 1-4 (config 5 = config 3 through the offload engine); "L" = operator count
# scaled so that the totals BASELINE.json states are reached.
CONFIGS = {
    "1": dict(D=256, S=12, M=2, N0=4, n_ops=1, n_site=0, dims="multinomial",
              rules=np.array([(1, 1)], dtype=np.int32)),
    "2": dict(D=2048, S=100, M=8, N0=20, n_ops=256, n_site=4, dims="multinomial"),
    "3": dict(D=6000, S=250, M=12, N0=40, n_ops=2000, n_site=0, dims="lognormal", sigma=0.8),
    "4": dict(D=15400, S=400, M=16, N0=50, n_ops=1500, n_site=8, dims="lognormal", sigma=1.0),
    "3L": dict(D=6000, S=250, M=12, N0=40, n_ops=10000, n_site=0, dims="lognormal", sigma=0.8),
    "4L": dict(D=15400, S=400, M=16, N0=50, n_ops=9000, n_site=8, dims="lognormal", sigma=1.0),
}
_SEED_OF = {"1": 1, "2": 2, "3": 3, "4": 4, "3L": 3, "4L": 4}


def make_config(cfg: str, n_ops: int | None = None, **over) -> BlockSparseSet:
    """BASELINE.json config by name ('1','2','3','4','3L','4L'); seed = BASE_SEED + config number."""
    kw = dict(CONFIGS[cfg])
    if n_ops is not None:
        kw["n_ops"] = n_ops
    kw.update(over)
    return make_set(f"config{cfg}", BASE_SEED + _SEED_OF[cfg], **kw)
