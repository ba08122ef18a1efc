"""Host logic of the tcgen05 GEMV's row-exact work split (csrc/gemv_umma.cuh, include/dovetail_hooks.h
dovetail_hooks_umma_tables), checked on the CPU against an independent statement of the dealing rule
(csrc/gemv.cuh GemvGroup: contiguous unit ranges differing by at most one unit; gate / up rows paired; QKV rows
dealt as rotary pairs (i, i + head_dim / 2)): every virtual row of every CTA sits at a tile position whose 8-row box
really starts at that row's matrix / row minus its offset in the box, positions are unique, super-blocks hold at
most 16 boxes, and the CTAs together cover every row of every matrix exactly once."""
import numpy as np
import pytest

from paper_2412_18934_b200 import binding, build


def virtual_rows(rows, paired, pairperm, ctas, c):
    """(matrix, row) of the virtual rows 0 .. cnt-1 of CTA c, from the rule alone."""
    tot = sum(rows)
    units = rows[0] if paired else tot // (2 if pairperm else 1)
    base, rem = divmod(units, ctas)
    u0, un = c * base + min(c, rem), base + (1 if c < rem else 0)
    out = []
    if paired:
        for j in range(len(rows)):
            out += [(j, u0 + i) for i in range(un)]
        return out
    unit = 2 if pairperm else 1
    for g in range(u0 * unit, (u0 + un) * unit):
        if pairperm:  # virtual order (0, dh/2, 1, dh/2 + 1, ...) inside every head of the concatenated rows
            w = g % pairperm
            g = g - w + w // 2 + (w % 2) * (pairperm // 2)
        j = 0
        while g >= rows[j]:
            g -= rows[j]
            j += 1
        out.append((j, g))
    return out


CASES = [
    ([5120], 0, 0, 148),                     # O / down / DGF of the 13B shape: 34.6 rows per CTA
    ([5120, 5120, 5120], 0, 128, 148),       # QKV, 13B shape: rotary pairs across heads and matrices
    ([4096, 1024, 1024], 0, 128, 148),       # QKV with grouped-query attention (Llama-3-8B shape)
    ([13824, 13824], 1, 0, 148),             # gate / up paired: two super-blocks
    ([32000], 0, 0, 148),                    # LM head: 216.2 rows per CTA
    ([128256], 0, 0, 148),                   # LM head of a 128k vocabulary: 7 super-blocks
    ([192], 0, 0, 148), ([1000], 0, 0, 148), ([256, 128, 128], 0, 64, 148), ([320, 320], 1, 0, 148), ([5120], 0, 0, 74),
]


@pytest.mark.parametrize("rows,paired,pairperm,ctas", CASES)
def test_tables_place_every_row_in_a_box_that_holds_it(rows, paired, pairperm, ctas):
    build.build()
    t = binding.dovetail_hooks_umma_tables(rows, paired, pairperm, ctas)
    seen = [np.zeros(r, np.int32) for r in rows]
    for c in range(ctas):
        want = virtual_rows(rows, paired, pairperm, ctas, c)
        assert t["cnt"][c] == len(want)
        n_sb = int(t["n_sb"][c])
        if not want:
            assert n_sb == 0
            continue
        ng = t["n_grp"][c][:n_sb]
        total = int(ng.sum())
        per = -(-total // n_sb)  # boxes per super-block: the fewest super-blocks, filled evenly, the last takes the rest
        assert n_sb == -(-total // 16) and per <= 16 and (ng[:-1] == per).all() and 1 <= ng[-1] <= per
        assert (t["n_grp"][c][n_sb:] == 0).all()
        pos = t["vpos"][c][:len(want)].astype(np.int64)
        assert len(set(pos.tolist())) == len(want), "two virtual rows share a tile position"
        for v, (j, n) in enumerate(want):
            sb, trow = int(pos[v]) >> 7, int(pos[v]) & 127
            g, r = trow >> 3, trow & 7
            assert sb < n_sb and g < ng[sb]
            code = int(t["grp"][c][sb][g])
            assert (code >> 28, (code & 0x0fffffff) + r) == (j, n), f"cta {c} virtual row {v}"
            seen[j][n] += 1
    for j, s in enumerate(seen):
        assert (s == 1).all(), f"matrix {j}: rows covered {np.unique(s)} times"


def test_too_many_super_blocks_is_refused():
    with pytest.raises(binding.DovetailError) as e:
        binding.dovetail_hooks_umma_tables([400000], 0, 0, 148)  # 2703 rows per CTA: 22 super-blocks > 8
    assert e.value.code == binding.ECAPACITY
