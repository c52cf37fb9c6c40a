"""Shared comparison helpers for the GPU parity tests (gates from BASELINE.json north_star)."""
import numpy as np

import oracle

L2_GATE = 1e-5          # per-energy image relative L2 error
PIX_GATE = 1e-3         # per-pixel relative error wherever I_ref >= 1e-6 max(I_ref)
PIX_FLOOR = 1e-6


def oracle_run(w, linear=False, **kw):
    return oracle.run(w.materials, w.voxel_nm, w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp,
                      w.angles, w.ewald, linear=linear, **kw)


def compare(out_gpu, cnt_gpu, out_ref, cnt_ref, label=""):
    """Returns a dict of error measures after asserting the north_star gates per energy."""
    out_gpu = np.asarray(out_gpu, np.float64)
    res = {"l2": [], "pix": [], "l2_nocentre": []}
    for e in range(out_ref.shape[0]):
        ref, got = out_ref[e], out_gpu[e]
        assert np.isfinite(got).all(), f"{label} e={e}: non-finite output"
        if cnt_gpu is not None:
            bad = int((np.asarray(cnt_gpu[e]) != cnt_ref[e]).sum())
            assert bad == 0, f"{label} e={e}: {bad} pixels differ in valid-angle count"
        l2 = np.linalg.norm(got - ref) / np.linalg.norm(ref)
        mask = ref >= PIX_FLOOR * ref.max()
        pix = (np.abs(got - ref)[mask] / ref[mask]).max()
        cy, cx = ref.shape[0] // 2, ref.shape[1] // 2
        r2, g2 = ref.copy(), got.copy()
        r2[cy - 1:cy + 2, cx - 1:cx + 2] = 0; g2[cy - 1:cy + 2, cx - 1:cx + 2] = 0
        l2n = np.linalg.norm(g2 - r2) / max(np.linalg.norm(r2), 1e-300)
        res["l2"].append(l2); res["pix"].append(pix); res["l2_nocentre"].append(l2n)
        assert l2 <= L2_GATE, f"{label} e={e}: relative L2 {l2:.3e} > {L2_GATE}"
        assert pix <= PIX_GATE, f"{label} e={e}: per-pixel relative error {pix:.3e} > {PIX_GATE} ({mask.sum()} px gated)"
        assert (got[cnt_ref[e] == 0] == 0).all(), f"{label} e={e}: never-valid pixels must be 0"
    return res
