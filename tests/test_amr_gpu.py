"""GPU parity of NEXT-3 (two-level static refinement) through the C ABI: z4c_restrict,
z4c_prolongate and z4c_two_level_step against the oracle's operators element by element.
Tolerances: the interpolation is bit-specified (reading R-I1: exact dyadic weights, difference-from-reference sum in
a fixed order, every operation rounded separately), so both operators are compared BIT FOR BIT; two-level steps: the
hot path's 1e-12 (one step) / 1e-10 (many steps) of max(|field|_max, S)."""
from dataclasses import replace

import numpy as np
import pytest

from paper_2409_10383_b200 import inputs as I
from tests.parity import perturbation_scale, rel_err

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Z():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2409_10383_b200 import build, z4c
    build.build()
    return z4c


def levels(Z, pc, pf, uc, uf):
    coarse = Z.Z4c(pc)
    fine = Z.Z4c(pf, stream=coarse.stream)           # both levels on one stream (the ABI requires it)
    coarse.set_initial_data(uc)
    fine.set_initial_data(uf)
    return coarse, fine


def padded(sim):
    sim.sync()
    return sim.state.cpu().numpy()


CASES = {
    # (coarse n, coarse nb, bc, fine n, fine nb, origin, ng)
    "corner_periodic": (16, (2, 2, 2), 0, 16, (2, 2, 2), (0, 0, 0), 3),
    "inner_box_outflow": (12, (2, 2, 2), 1, 8, (2, 1, 3), (7, 10, 3), 3),
    "straddles_blocks_periodic": (8, (3, 2, 2), 0, 8, (2, 2, 1), (8, 5, 6), 3),    # box not aligned with coarse blocks
    "o6_corner": (16, (2, 2, 1), 0, 16, (2, 1, 1), (16, 8, 0), 4),
}


@pytest.mark.parametrize("name", list(CASES))
def test_restrict_and_prolongate_against_the_oracle(Z, oracle, name):
    nc, nbc, bc, nf, nbf, origin, ng = CASES[name]
    pc = replace(I.params_noise(nc, nbc, dx=0.1), bc=bc, ng=ng)
    pf = replace(pc, n=nf, nb=nbf, dx=0.05, bc=1)
    uc = I.smooth_random_data(pc, 3, 0.1)
    uf = I.smooth_random_data(pf, 4, 0.1)                               # unrelated data: nothing cancels by accident
    coarse, fine = levels(Z, pc, pf, uc, uf)
    uc_e, uf_e = coarse.get_interior(), fine.get_interior()              # after the library's own enforcement
    fine_before = padded(fine)
    # --- restriction -------------------------------------------------------------------------------------
    fine.restrict_to(coarse, origin)
    got = coarse.get_interior()
    want = uc_e.copy()
    R = oracle.restrict(uf_e, ng, nf)
    Mz, My, Mx = R.shape[1:]
    want[:, origin[2]:origin[2] + Mz, origin[1]:origin[1] + My, origin[0]:origin[0] + Mx] = R
    assert np.array_equal(got, want)
    untouched = np.ones(want.shape[1:], bool)
    untouched[origin[2]:origin[2] + Mz, origin[1]:origin[1] + My, origin[0]:origin[0] + Mx] = False
    assert np.array_equal(got[:, untouched], uc_e[:, untouched])          # nothing else is written
    from tests.parity import padded_reference
    assert np.array_equal(padded(coarse), padded_reference(got, pc))      # the coarse ghosts were refilled (O2)
    # --- prolongation ------------------------------------------------------------------------------------
    fine.prolongate_from(coarse, origin)
    after = padded(fine)
    Nf = pf.N
    lo, hi = (-ng,) * 3, (Nf[0] + ng, Nf[1] + ng, Nf[2] + ng)
    box = oracle.prolong(got, ng, bc, origin, lo, hi)                     # the whole padded fine region
    m = nf + 2 * ng
    checked = 0
    for bz in range(nbf[2]):
        for by in range(nbf[1]):
            for bx in range(nbf[0]):
                b = (bz * nbf[1] + by) * nbf[0] + bx
                ref = box[:, bz * nf:bz * nf + m, by * nf:by * nf + m, bx * nf:bx * nf + m]
                gz, gy, gx = np.meshgrid(np.arange(m) + bz * nf - ng, np.arange(m) + by * nf - ng,
                                         np.arange(m) + bx * nf - ng, indexing="ij")
                outside = (gx < 0) | (gx >= Nf[0]) | (gy < 0) | (gy >= Nf[1]) | (gz < 0) | (gz >= Nf[2])
                assert np.array_equal(after[:, b][:, outside], ref[:, outside])
                assert np.array_equal(after[:, b][:, ~outside], fine_before[:, b][:, ~outside])   # left alone
                checked += int(outside.sum())
    assert checked > 0
    coarse.close()
    fine.close()


@pytest.mark.parametrize("mode", [2, 1])
def test_two_level_steps_against_the_oracle(Z, oracle, mode):
    """The refined-corner wave of PAPER.md:171 on BASELINE's wave: coarse 32^3 in 8 blocks of 16^3, the corner block
    refined once (8 fine blocks of 16^3), one dt; 1 step at 1e-12, 12 steps at 1e-10, both levels. mode 2: the fused
    stage kernel per level and stage (state ping-pong), mode 1: RHS + update-with-push in place."""
    pc = replace(I.params_linear_wave(32, 16), cfl=0.125)
    pf = replace(pc, nb=(2, 2, 2), dx=pc.dx / 2, cfl=0.25, bc=1)
    uc, uf = I.linear_wave_data(pc), I.linear_wave_data(pf)
    coarse, fine = levels(Z, pc, pf, uc, uf)
    for s in (coarse, fine):
        s.set_fused(mode)
        assert s.effective_mode()[1] == mode
    rc, rf = oracle.enforce(pc, uc)[0], oracle.enforce(pf, uf)[0]
    done = 0
    for target, tol in ((1, 1e-12), (12, 1e-10)):
        rc, rf, bad = oracle.step_two_level(pc, pf, 16, (0, 0, 0), rc, rf, target - done)
        assert bad == 0
        fine.two_level_step(coarse, (0, 0, 0), target - done)
        done = target
        for sim, ref, p in ((coarse, rc, pc), (fine, rf, pf)):
            sim.sync()
            err = rel_err(sim.get_interior(), ref, perturbation_scale(ref, p))
            assert err.max() <= tol, (target, dict(zip(I.FIELD_NAMES, err)))
    assert abs(coarse.time() - fine.time()) < 1e-15 and abs(fine.time() - 12 * pf.dt) < 1e-15
    # the same on strong-field data with an off-corner box (all nonlinear terms, both upwind sides), one step
    pc2 = replace(I.params_noise(16, (2, 2, 2), dx=0.1), cfl=0.125)
    pf2 = replace(pc2, n=8, nb=(2, 3, 2), dx=0.05, cfl=0.25, bc=1)
    o = (9, 4, 16)
    u2c = I.smooth_random_data(pc2, 7, 0.05)
    # fine data = the coarse field interpolated onto the fine box (by the oracle), so the levels start consistent
    u2f = oracle.prolong(oracle.enforce(pc2, u2c)[0], 3, pc2.bc, o, (0, 0, 0), pf2.N)
    c2, f2 = levels(Z, pc2, pf2, u2c, u2f)
    for s in (c2, f2):
        s.set_fused(mode)
    rc2, rf2, bad = oracle.step_two_level(pc2, pf2, 8, o, oracle.enforce(pc2, u2c)[0], oracle.enforce(pf2, u2f)[0], 1)
    assert bad == 0
    f2.two_level_step(c2, o, 1)
    for sim, ref, p in ((c2, rc2, pc2), (f2, rf2, pf2)):
        sim.sync()
        err = rel_err(sim.get_interior(), ref, perturbation_scale(ref, p))
        assert err.max() <= 1e-12, dict(zip(I.FIELD_NAMES, err))
    for s in (coarse, fine, c2, f2):
        s.close()


def test_two_level_argument_checks(Z):
    pc = replace(I.params_linear_wave(32, 16), cfl=0.125)
    pf = replace(pc, nb=(2, 2, 2), dx=pc.dx / 2, cfl=0.25, bc=1)
    coarse = Z.Z4c(pc)
    fine = Z.Z4c(pf, stream=coarse.stream)
    other = Z.Z4c(pf)                                                   # its own stream
    with pytest.raises(Z.Z4cError):
        other.restrict_to(coarse, (0, 0, 0))
    with pytest.raises(Z.Z4cError):
        fine.restrict_to(coarse, (20, 0, 0))                            # box leaves the coarse mesh
    bad_dx = Z.Z4c(replace(pf, dx=pc.dx / 3), stream=coarse.stream)
    with pytest.raises(Z.Z4cError):
        bad_dx.prolongate_from(coarse, (0, 0, 0))
    bad_dt = Z.Z4c(replace(pf, cfl=0.2), stream=coarse.stream)
    with pytest.raises(Z.Z4cError):
        bad_dt.two_level_step(coarse, (0, 0, 0), 1)
    for s in (coarse, fine, other, bad_dx, bad_dt):
        s.close()


def test_two_level_step_with_four_ghosts(Z, oracle):
    """The paper's production scheme on the refined-corner wave: 4 ghosts, 6th-order stencils, 5-node interpolation
    ("5th order for 4 ghost"), 2 steps, both levels at 1e-12."""
    pc = replace(I.params_linear_wave(32, 16), cfl=0.125, ng=4)
    pf = replace(pc, nb=(2, 2, 2), dx=pc.dx / 2, cfl=0.25, bc=1)
    uc, uf = I.linear_wave_data(pc), I.linear_wave_data(pf)
    coarse, fine = levels(Z, pc, pf, uc, uf)
    rc, rf, bad = oracle.step_two_level(pc, pf, 16, (0, 0, 0), oracle.enforce(pc, uc)[0], oracle.enforce(pf, uf)[0], 2)
    assert bad == 0
    fine.two_level_step(coarse, (0, 0, 0), 2)
    for sim, ref, p in ((coarse, rc, pc), (fine, rf, pf)):
        sim.sync()
        err = rel_err(sim.get_interior(), ref, perturbation_scale(ref, p))
        assert err.max() <= 1e-12, dict(zip(I.FIELD_NAMES, err))
    coarse.close()
    fine.close()


def _padded_box_from_interior(u, p, b3):
    """Padded box [F][m][m][m] of block b3 = (bx, by, bz) by O2's definition (periodic wrap) from the global interior."""
    n, g = p.n, p.ng
    idx = [(np.arange(-g, n + g) + b * n) % N for b, N in zip(b3, p.N)]
    return u[:, idx[2][:, None, None], idx[1][None, :, None], idx[0][None, None, :]]


def test_two_level_bench_workload_at_full_size(Z, oracle):
    """The workload `bench.py --workload two_level_wave_256` times, in its launch configuration (both packs in mode 2:
    fused stage kernel per level, exchange on the buffer just written; 512 + 512 blocks of 32^3), after two steps, on
    sampled outputs the oracle computes one by one -- all bit for bit, since the exchange is bit-specified (R-I1):
    covered coarse cells = oracle restriction of the fine blocks above them; coarse ghosts = images of the interior
    (written by k_restrict for the cells it changed); fine ghosts outside the box = oracle prolongation of the coarse
    interior (faces, edges, corners of the box); fine ghosts inside the box = the neighbouring fine block's cells.
    Seeded 1e-10 noise on top of the x-directed wave makes every cell distinct, so a wrong y / z index cannot hide."""
    import bench
    import torch
    pc, pf, origin = bench.two_level_workload()
    uc0 = I.linear_wave_data(pc) + I.noise_data(pc, 31)
    uf0 = I.linear_wave_data(pf) + I.noise_data(pf, 32)
    coarse, fine = levels(Z, pc, pf, uc0, uf0)
    del uc0, uf0
    assert coarse.effective_mode()[1] == 2 and fine.effective_mode()[1] == 2
    fine.two_level_step(coarse, origin, 2)
    coarse.sync()
    uc, uf = coarse.get_interior(), fine.get_interior()
    assert np.all(np.isfinite(uc)) and np.all(np.isfinite(uf))
    n, g, h = pc.n, pc.ng, pc.n // 2
    # (i) restriction: coarse cells under sampled fine blocks (corner, far corner, inside, on a face of the box)
    for bx, by, bz in ((0, 0, 0), (7, 7, 7), (3, 4, 5), (7, 0, 3)):
        sub = uf[:, bz * n:(bz + 1) * n, by * n:(by + 1) * n, bx * n:(bx + 1) * n]
        want = oracle.restrict(sub, g, n)
        got = uc[:, origin[2] + bz * h:origin[2] + (bz + 1) * h, origin[1] + by * h:origin[1] + (by + 1) * h,
                 origin[0] + bx * h:origin[0] + (bx + 1) * h]
        assert np.array_equal(got, want), (bx, by, bz)
    # (ii) coarse ghosts, blocks next to / inside / far from the box and across the periodic faces
    for b3 in ((1, 2, 2), (2, 2, 2), (5, 6, 1), (0, 0, 0), (7, 7, 7), (4, 4, 4)):
        b = (b3[2] * pc.nb[1] + b3[1]) * pc.nb[0] + b3[0]
        assert np.array_equal(coarse.state[:, b].cpu().numpy(), _padded_box_from_interior(uc, pc, b3)), b3
    # (iii) prolongation: windows of the shell around the fine region (indices relative to its corner)
    Nf = pf.N[0]
    windows = (((-g, 100, 100), (0, 140, 140)), ((Nf, 30, 200), (Nf + g, 70, 256)), ((90, -g, 10), (130, 0, 40)),
               ((10, Nf, 10), (60, Nf + g, 40)), ((120, 120, -g), (136, 136, 0)), ((0, 224, Nf), (40, 256, Nf + g)),
               ((-g, -g, -g), (0, 0, 0)), ((Nf, Nf, Nf), (Nf + g, Nf + g, Nf + g)), ((Nf, -g, 60), (Nf + g, 0, 68)),
               ((-g, 28, Nf), (0, 36, Nf + g)))
    state_f = fine.state
    for lo, hi in windows:
        want = oracle.prolong(uc, g, pc.bc, origin, lo, hi)
        ax = []
        for d in range(3):                                   # a block whose padded box holds each index, and where
            c = np.arange(lo[d], hi[d])
            bd = np.clip(c // n, 0, pf.nb[d] - 1)
            ax.append((bd, c - bd * n + g))
        (bxs, lxs), (bys, lys), (bzs, lzs) = ax
        blk = (bzs[:, None, None] * pf.nb[1] + bys[None, :, None]) * pf.nb[0] + bxs[None, None, :]
        got = state_f[:, torch.from_numpy(blk).to(state_f.device),
                      torch.from_numpy(np.broadcast_to(lzs[:, None, None], blk.shape).copy()).to(state_f.device),
                      torch.from_numpy(np.broadcast_to(lys[None, :, None], blk.shape).copy()).to(state_f.device),
                      torch.from_numpy(np.broadcast_to(lxs[None, None, :], blk.shape).copy()).to(state_f.device)]
        assert np.array_equal(got.cpu().numpy(), want), (lo, hi)
    # (iv) fine ghosts inside the box: an inner block's padded box is a window of the fine interior
    for b3 in ((3, 4, 5), (1, 1, 6)):
        b = (b3[2] * pf.nb[1] + b3[1]) * pf.nb[0] + b3[0]
        assert np.array_equal(state_f[:, b].cpu().numpy(), _padded_box_from_interior(uf, pf, b3)), b3
    coarse.close()
    fine.close()
