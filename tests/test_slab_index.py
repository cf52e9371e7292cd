"""Index algebra of the row-pass twiddle slab (csrc/fenc_device.cuh: tw_slab_fill, tile_round_ct<..., TWS = 2>), modelled in
Python (host logic, no GPU): for every thread, round, stage and twiddle slot, the slab entry a round reads was filled from the
table entry the same round reads when it indexes the table directly.  A wrong level offset, a wrong transposition or an
off-by-one in the heap order fails here; the GPU parity tests then confirm the kernels."""
import pytest

LT = 10                     # FENC_ROW_LT: 2^10 contiguous coefficients per row tile
T, NT8 = 1 << LT, 1 << (LT - 3)
ROUNDS_FWD = [(5, (0, 1, 2)), (2, (0, 1, 2)), (0, (0, 1))]   # (PW, active stages) of tile_rounds_ct<FWD, LO = 0, NB = 8>
ROUNDS_INV = [(0, (0, 1, 2)), (3, (0, 1, 2)), (6, (0, 1))]   # inverse: low bits first


def slab_fill(logN, tile):
    """slab position -> table index, as tw_slab_fill copies them"""
    base = (1 << logN) + (tile << LT)
    slab = {}
    for idx in range(1, T):
        lvl = idx.bit_length() - 1
        loc = idx - (1 << lvl)
        if lvl == LT - 1:
            pos = (4 + (loc & 3)) * NT8 + (loc >> 2)
        elif lvl == LT - 2:
            pos = (2 + (loc & 1)) * NT8 + (loc >> 1)
        else:
            pos = idx
        assert pos not in slab, "two table entries land on one slab slot"
        slab[pos] = (base >> (LT - lvl)) + loc
    return slab


def round_reads(PW, stages, tid, logN_geo, tile, transposed):
    """[(stage, slot i, index read)] of one thread in one round: the table index formula of tile_round_ct with the geometry
    (logN_geo, tile) of a contiguous row tile; transposed: the TWS = 2, PW = 0 addressing of the two lowest levels"""
    ebase = ((tid >> PW) << (PW + 3)) | (tid & ((1 << PW) - 1))
    nj = (1 << logN_geo) + (tile << LT) + ebase
    out = []
    for s in stages:
        for i in range(1 << (2 - s)):
            if transposed and PW == 0 and s == 1:
                out.append((s, i, (2 + i) * NT8 + tid))
            elif transposed and PW == 0 and s == 0:
                out.append((s, i, (4 + i) * NT8 + tid))
            else:
                out.append((s, i, (nj >> (PW + s + 1)) + i))
    return out


@pytest.mark.parametrize("logN", [12, 14, 16])
@pytest.mark.parametrize("rounds", [ROUNDS_FWD, ROUNDS_INV])
def test_slab_reads_equal_table_reads(logN, rounds):
    for tile in {0, 1, (1 << (logN - LT)) - 1}:
        slab = slab_fill(logN, tile)
        for PW, stages in rounds:
            for tid in range(NT8):
                direct = round_reads(PW, stages, tid, logN, tile, transposed=False)      # the table, global geometry
                via = round_reads(PW, stages, tid, LT, 0, transposed=True)               # the slab, row_slab_geo()
                assert [(s, i) for s, i, _ in direct] == [(s, i) for s, i, _ in via]
                for (s, i, g), (_, _, p) in zip(direct, via):
                    assert slab[p] == g, (logN, tile, PW, s, i, tid)


def test_transposed_levels_are_unit_stride():
    """the point of the transposition: in the round over the lowest bits consecutive threads read consecutive slab entries"""
    for s in (0, 1):
        for i in range(1 << (2 - s)):
            idx = [next(p for ss, ii, p in round_reads(0, (0, 1), tid, LT, 0, True) if (ss, ii) == (s, i)) for tid in range(NT8)]
            assert idx == list(range(idx[0], idx[0] + NT8))


def test_column_pass_twiddles_fit_the_staged_256_entries():
    """fused column kernel (TWS = 1): a target's forward column stages read tw[1 .. 255] only, whatever the column tile"""
    logN, brow, LC, LTc = 16, 8, 2, 10
    for tile in (0, 5, 63):
        for PW, stages in [(7, (0, 1, 2)), (4, (0, 1, 2)), (2, (0, 1))]:
            gpw = PW - LC + brow
            for tid in range(1 << (LTc - 3)):
                ebase = ((tid >> PW) << (PW + 3)) | (tid & ((1 << PW) - 1))
                gidx = ((ebase >> LC) << brow) | (tile << LC) | (ebase & ((1 << LC) - 1))
                nj = (1 << logN) + gidx
                for s in stages:
                    for i in range(1 << (2 - s)):
                        assert 1 <= (nj >> (gpw + s + 1)) + i <= 255


def test_first_round_order_covers_the_tile_in_coalesced_runs():
    """REGIN (row kernels, slab form): thread tid loads element round_ebase<PW0>(tid) + (i << PW0), PW0 = 5 for the forward
    row pass -- every element of the tile exactly once, 32 consecutive words per warp and i, and exactly the elements the
    first round (window PW0) gives that thread."""
    PW0 = ROUNDS_FWD[0][0]
    seen = set()
    for tid in range(NT8):
        eb = ((tid >> PW0) << (PW0 + 3)) | (tid & ((1 << PW0) - 1))
        for i in range(8):
            seen.add(eb + (i << PW0))
    assert seen == set(range(T))
    for warp in range(NT8 // 32):
        for i in range(8):
            run = [(((t >> PW0) << (PW0 + 3)) | (t & ((1 << PW0) - 1))) + (i << PW0) for t in range(32 * warp, 32 * warp + 32)]
            assert run == list(range(run[0], run[0] + 32))
