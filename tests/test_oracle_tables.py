"""Pins for the oracle's integer tables (S0): brute force and counting identities."""
import numpy as np
import pytest

import oracle
from paper_1808_10375_b200 import synth


@pytest.mark.parametrize("cfg_i,ny,nx,th,tw", [(0, 10, 10, 8, 32), (1, 5, 4, 8, 32), (0, 4, 5, 16, 16), (3, 2, 3, 8, 32)])
def test_coverage_lists_bruteforce_and_identities(cfg_i, ny, nx, th, tw):
    cfg = synth.CONFIGS[cfg_i].scaled(ny, nx)
    pos = synth.make_positions(cfg, np.random.default_rng(0))
    N, H, W = cfg.N, cfg.obj_h, cfg.obj_w
    ptr, views = oracle.coverage(N, pos, H, W, th, tw)
    nty, ntx = -(-H // th), -(-W // tw)
    assert ptr[0] == 0 and ptr[-1] == len(views) and len(ptr) == nty * ntx + 1
    # per-pixel brute force: a view is in a tile's list iff it covers at least one pixel of the tile
    cover = np.zeros((cfg.n_views, H, W), bool)
    for j, (y, x) in enumerate(pos):
        cover[j, y:y + N, x:x + N] = True
    for ty in range(nty):
        for tx in range(ntx):
            lst = views[ptr[ty * ntx + tx]:ptr[ty * ntx + tx + 1]]
            want = np.nonzero(cover[:, ty * th:(ty + 1) * th, tx * tw:(tx + 1) * tw].any(axis=(1, 2)))[0]
            assert np.array_equal(lst, want)
            assert np.all(np.diff(lst) > 0)                      # strictly ascending
    # each view appears in exactly (#tile rows it touches) * (#tile cols it touches) lists
    per_view = np.bincount(views, minlength=cfg.n_views)
    want = ((pos[:, 0] + N - 1) // th - pos[:, 0] // th + 1) * ((pos[:, 1] + N - 1) // tw - pos[:, 1] // tw + 1)
    assert np.array_equal(per_view, want)


def test_cover_count_and_window_table():
    cfg = synth.CONFIGS[0]
    pos = synth.make_positions(cfg, np.random.default_rng(0))
    cnt = oracle.cover_count(cfg.N, pos, cfg.obj_h, cfg.obj_w)
    assert cnt.sum() == cfg.n_views * cfg.N ** 2
    want = np.zeros_like(cnt)
    for y, x in pos:
        want[y:y + cfg.N, x:x + cfg.N] += 1
    assert np.array_equal(cnt, want)
    wt = oracle.window_table(pos, cfg.obj_w)
    assert np.array_equal(wt[:, :2], pos)
    assert np.array_equal(wt[:, 2], pos[:, 0] * cfg.obj_w + pos[:, 1])
