"""Host logic of the slice-sweep kernel's launch plan (no GPU): the block -> (tile, t-segment) index function the kernel
evaluates (csrc/fine_sweep.cuh sweep_block_coords, the same code compiled for the host) covers every (tile, slice) of the
lattice exactly once, whatever the tail split chosen by the schedule simulation."""
import numpy as np
import pytest

import paper_2211_13719_b200 as mrhs

CASES = [
    ([48, 48, 48, 48], 12, mrhs.FULL, 148),   # the bench workload: 3456 tiles, the last 52 cut in two
    ([48, 48, 48, 48], 12, mrhs.ODD, 148),
    ([48, 48, 48, 48], 24, mrhs.EVEN, 148),
    ([24, 24, 24, 24], 12, mrhs.FULL, 148),
    ([24, 24, 24, 24], 48, mrhs.ODD, 148),
    ([32, 16, 8, 24], 4, mrhs.FULL, 148),
    ([16, 16, 16, 16], 24, mrhs.FULL, 132),    # another SM count
    ([8, 4, 4, 6], 12, mrhs.FULL, 148),        # fewer blocks than SMs: t-segments for all tiles
    ([48, 48, 48, 48], 12, mrhs.FULL, 7),      # a tiny device: many waves
]


@pytest.mark.parametrize("dims,nrhs,parity,sms", CASES)
def test_blocks_cover_every_tile_slice_once(dims, nrhs, parity, sms):
    grid, threads, tiles, n_whole, tail_tiles, tail_seg, lt, cy, cz = mrhs.sweep_plan(dims, nrhs, parity, sms)
    X, Y, Z, T = dims
    xe = X if parity == mrhs.FULL else X // 2
    nxb = xe // mrhs.xblock(xe, nrhs)
    assert tiles == nxb * (Y // 2) * (Z // 2)
    assert threads % 32 == 0 and threads <= 512
    assert T % lt == 0 and (tail_tiles == 0 or (T % tail_seg == 0 and lt == T))
    assert grid == n_whole + tail_tiles * tail_seg
    assert n_whole == tiles * (T // lt) - tail_tiles
    cover = np.zeros((nxb, Y // 2, Z // 2, T), dtype=np.int32)
    for b, (xb, y0, z0, t0, n) in enumerate(mrhs.sweep_blocks(dims, nrhs, parity, sms, 0, grid)):
        assert 0 <= xb < nxb and y0 % 2 == 0 and z0 % 2 == 0 and 0 <= y0 < Y and 0 <= z0 < Z
        assert 0 <= t0 and t0 + n <= T
        assert n == (lt if b < n_whole else T // tail_seg)
        cover[xb, y0 // 2, z0 // 2, t0:t0 + n] += 1
    assert cover.min() == 1 and cover.max() == 1


def test_tail_split_shortens_the_last_wave():
    """48^4, N_rhs = 12 on 148 SMs: 3456 whole-line tiles are 23.35 waves; the plan cuts the leftover tiles so that the
    blocks of the last wave are short ones, and never splits when the grid fills whole waves."""
    grid, _, tiles, n_whole, tail_tiles, tail_seg, lt, _, _ = mrhs.sweep_plan([48] * 4, 12, mrhs.FULL, 148)
    assert lt == 48 and tail_tiles > 0 and tail_seg >= 2
    assert n_whole % 148 == 0 or tail_tiles * tail_seg >= 148 - n_whole % 148
    # 3456 tiles on 144 SMs are exactly 24 waves: nothing to balance
    assert mrhs.sweep_plan([48] * 4, 12, mrhs.FULL, 144)[4] == 0


def test_plan_argument_errors():
    with pytest.raises(mrhs.MrhsError) as e:
        mrhs.sweep_plan([48] * 4, 3, mrhs.FULL, 148)          # odd N_rhs: no sweep kernel
    assert e.value.status == mrhs.ERR_UNSUPPORTED
    with pytest.raises(mrhs.MrhsError):
        mrhs.sweep_plan([48, 48, 47, 48], 12, mrhs.FULL, 148)
    with pytest.raises(mrhs.MrhsError):
        mrhs.sweep_blocks([8, 4, 4, 6], 12, mrhs.FULL, 148, 10 ** 6, 1)
