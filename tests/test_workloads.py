"""The seeded input generator: recipe of SURVEY §8(d) / DESIGN.md "Input recipe"."""
import numpy as np
import pytest

import workloads as W
from workloads.values import block_values, splitmix64_at


def test_splitmix64_published_vectors():
    # first outputs of SplitMix64 for seed 1234567 (the reference C implementation's well-known vector)
    got = [int(x) for x in splitmix64_at(1234567, np.arange(5))]
    assert got == [6457827717110365317, 3203168211198807973, 9817491932198370423,
                   4593380528125082431, 16408922859458223821]


def test_values_uniform_deterministic_and_keyed_by_block_and_element():
    v = block_values(7, np.array([3, 4]), np.array([5, 2]))
    assert v.shape == (7,) and (v >= -1).all() and (v < 1).all()
    assert (block_values(7, np.array([4]), np.array([2])) == v[5:]).all()
    assert (block_values(7, np.array([3]), np.array([5])) == v[:5]).all()
    assert not (block_values(8, np.array([3]), np.array([5])) == v[:5]).any()
    big = block_values(1, np.array([0]), np.array([200000]))
    assert abs(big.mean()) < 0.01 and abs(big.var() - 1 / 3) < 0.01


def test_label_grid_config1():
    g = W.label_grid(12, 2, 4)
    assert g.tolist() == [[4, -2], [4, 0], [4, 2], [5, -1], [5, 1], [6, -2], [6, 0], [6, 2], [7, -1], [7, 1],
                          [8, -2], [8, 0]]
    assert len(W.selection_rules()) == 13
    assert all((int(r[0]) - int(r[1])) % 2 == 0 for r in W.selection_rules())


@pytest.mark.parametrize("cfg,T,B", [("1", 1, 7), ("2", 260, None), ("3", 2000, None)])
def test_config_shapes(cfg, T, B):
    s = W.make_config(cfg)
    assert s.n_tensors == T
    if B is not None:
        assert s.n_blocks == B
    assert int(s.meta["bond_dims"].sum()) == s.meta["D"] and s.meta["bond_dims"].min() >= 1
    # tensor records partition the block table
    assert s.tensors["first_block"][0] == 0
    assert (s.tensors["first_block"][1:] == np.cumsum(s.tensors["n_blocks"])[:-1]).all()
    assert int(s.tensors["n_blocks"].sum()) == s.n_blocks
    # conservation: sum_k sign_k qn_k == dq, block by block
    t_of_b = np.repeat(np.arange(T), s.tensors["n_blocks"])
    sign = s.tensors["sign"][t_of_b][:, :3].astype(np.int64)
    acc = (sign[:, :, None] * s.qn.astype(np.int64)).sum(axis=1)
    assert (acc == s.tensors["dq"][t_of_b]).all()
    # unused legs
    r2 = s.tensors["rank"][t_of_b] == 2
    assert (s.dim[r2, 2] == 1).all() and (s.qn[r2, 2] == 0).all()
    # placement: 512-aligned, disjoint, scattered
    assert (s.pool_off % 512 == 0).all()
    order = np.argsort(s.pool_off, kind="stable")
    ends = s.pool_off[order] + s.nelems[order] * 8
    assert (ends[:-1] <= s.pool_off[order][1:]).all() and int(ends[-1]) <= s.pool_bytes
    if s.n_blocks > 100:
        assert not (order == np.arange(s.n_blocks)).all()


def test_config2_has_rank3_site_tensors_with_local_leg():
    s = W.make_config("2")
    site = s.tensors[s.tensors["rank"] == 3]
    assert len(site) == 4
    b0 = int(site["first_block"][0])
    assert (s.dim[b0:, 1] == 1).all()
    loc = {tuple(x) for x in s.qn[b0:, 1].tolist()}
    assert loc == {(0, 0), (1, 1), (1, -1), (2, 0)}


def test_fill_pool_host_scattered_and_compact_agree():
    s = W.make_set("t", 3, D=64, S=10, M=2, N0=2, n_ops=13, n_site=1, dims="multinomial")
    pool, offs = W.fill_pool_host(s, chunk_elems=1000)
    cp, co = W.fill_pool_host(s, 5, 40, compact=True)
    ne = s.nelems
    for k, i in enumerate(range(5, 40)):
        a = pool[int(offs[i]) // 8: int(offs[i]) // 8 + int(ne[i])]
        b = cp[int(co[k]) // 8: int(co[k]) // 8 + int(ne[i])]
        assert (a == b).all()
        assert (a == block_values(s.seed, np.array([i]), np.array([int(ne[i])]))).all()
