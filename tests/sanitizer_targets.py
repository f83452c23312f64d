"""Small invocations of the kernels whose synchronisation is the delicate part: a plain stress-and-compare
script (`python tests/sanitizer_targets.py` on a B200).  It was written as a compute-sanitizer target, but that
tool is closed on this pool (profiles/r02_compute_sanitizer_unavailable.txt), so NO race checker stands behind
these kernels: what this script and the -m gpu tests give is result comparison only -- every case below is
checked against another route or the oracle, repeated calls must agree bit for bit, and outputs are
NaN-prefilled so that a tile read before it was written shows.

(1) __graft_entry__.smoke(); (2) blink_grid_image on the shared-memory route with more snapshots than
CTAs, so every CTA of k_fused hands its chunk ring and its aliased line buffers from one snapshot to
the next (also with the correction factors riding in the chunks); (3) blink_grid on the ring route;
(4) blink_grid_image on the warp-per-transform route (k_img1024) with a ring of 2 slots of U for 6
snapshots, so pass A waits on pass B through the global counters; (5) blink_dynspec; (6) the residue-class
kernels: k_img1024r (producer / consumer warps over a ring of two tiles, CTAs changing snapshot mid-run) and
k_cols_res at 2048^2 (tiles leaving as bulk copies while the next unit is formed).  Each result is
checked against the two-call route so a silent corruption would also fail here.  Not collected by
pytest (no test_ prefix); the hand-over cases (2) are also -m gpu tests (test_every_fused_instance_against_oracle)."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import __graft_entry__  # noqa: E402
from paper_2405_13478_b200 import blink, synth  # noqa: E402


def main():
    __graft_entry__.smoke()
    # (2), (3): 60 x 3 = 180 snapshots of 128^2 over 148 CTAs
    w = synth.config_station(n_t=60, n_ch=3, n_pix=128)
    vis = torch.from_numpy(w.vis()).cuda()
    plan = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, options=dict(grid_ring_min_snap=1))
    assert plan.query_i32(blink.Q_FUSED_PATH) == 1
    img = plan.grid_image(vis)
    ref = plan.image(plan.grid(vis))
    peak = ref.abs().amax(dim=(-2, -1), keepdim=True)
    assert ((img - ref).abs() <= 1e-5 * peak).all()
    rng = np.random.default_rng(1)
    gains = rng.uniform(0.5, 2.0, (w.n_ch, w.n_ant)) * np.exp(1j * rng.uniform(-3, 3, (w.n_ch, w.n_ant)))
    plan.set_corrections(gains, rng.uniform(0, 100, w.n_ant), 0.1, 0.2)
    two = plan.grid_image(plan.correct(vis))
    plan.apply_corrections(True)
    one = plan.grid_image(vis)
    assert ((one - two).abs() <= 1e-5 * two.abs().amax(dim=(-2, -1), keepdim=True)).all()
    dyn = plan.dynspec(img, 0.25)
    assert torch.isfinite(dyn).all()
    plan.close()
    # (4): k_img1024, 6 snapshots through a ring of 2
    w = synth.config_mwa1(n_t=3, n_ch=2)
    vis = torch.from_numpy(w.vis()).cuda()
    plan = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, options=dict(warp_route=2, warp_ring=2))
    assert plan.query_i32(blink.Q_FUSED_PATH) == 2
    img = plan.grid_image(vis)
    img = plan.grid_image(vis)                      # twice: the kernel must leave its counters zero
    plan0 = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, options=dict(warp_route=-1))
    ref = plan0.grid_image(vis)
    assert ((img - ref).abs() <= 1e-5 * ref.abs().amax(dim=(-2, -1), keepdim=True)).all()
    # (6): k_img1024r on the same six snapshots (384 units over 148 CTAs), then k_cols_res at 2048^2
    plan1 = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting)
    assert plan1.query_i32(blink.Q_WARP_KERNEL) == 2
    img = plan1.grid_image(vis)
    assert ((img - ref).abs() <= 1e-5 * ref.abs().amax(dim=(-2, -1), keepdim=True)).all()
    for pl in (plan, plan0, plan1):
        pl.close()
    w = synth.config_mwa2(n_t=1, n_ch=2)
    w.n_pix, w.pixscale = 2048, 30.0 * synth.ARCSEC
    vis = torch.from_numpy(w.vis()).cuda()
    plan = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting)
    assert plan.query_i32(blink.Q_WARP_KERNEL) == 3
    plan0 = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, options=dict(warp_route=-1))
    img, ref = plan.grid_image(vis), plan0.grid_image(vis)
    assert ((img - ref).abs() <= 1e-5 * ref.abs().amax(dim=(-2, -1), keepdim=True)).all()
    torch.cuda.synchronize()
    print("sanitizer targets ok")


if __name__ == "__main__":
    main()
