"""A numpy MODEL of the tensor route's arithmetic (no GPU): 3xTF32 operand split, one tensor-core add per K = 8 step
with a TRUNCATING fp32 accumulate, the fp32 epilogue (Eq. 2 derivative), the gradient contraction with its in-kernel
split of R and the fixed-order sum of the point segments.  It is neither the oracle nor the product: it exists to choose
between accumulator layouts on the CPU before a kernel is changed (VERDICT r1 next #3b).  It predicts the SHAPE of the
error (what scales with the number of adds into one accumulator); round 1's B200 measurements of the same plans were
2.4x larger than the model at both 256 and 384 dwell positions (6.9e-5 vs 2.9e-5, 1.0-1.4e-4 vs 5.3e-5), so the
hardware loses more per add than one truncation -- the ratios between layouts are what the model is used for."""
import numpy as np
import pytest

import gmco_cases as gc
import oracle


def tf32_rn(x):
    u = x.astype(np.float32).view(np.uint32).astype(np.uint64)
    return ((u + 0x1000) & 0xffffe000).astype(np.uint32).view(np.float32)        # cvt.rna.tf32.f32


def tf32_trunc(x):
    return (x.astype(np.float32).view(np.uint32) & np.uint32(0xffffe000)).view(np.float32)


def rz32(x64):
    y = x64.astype(np.float32)
    over = np.abs(y.astype(np.float64)) > np.abs(x64)
    return np.where(over, np.nextafter(y, np.float32(0)), y).astype(np.float32)


def mma(acc, a, b):
    """acc[M, N] (fp32) += a[M, 8] . b[8, N]: exact products and sum, ONE truncation into the fp32 accumulator."""
    return rz32(acc.astype(np.float64) + a.astype(np.float64) @ b.astype(np.float64))


def dose_model(D, T, layout):
    """D [N, A_pad], T [K, A_pad] fp32 -> dose [K, N] fp32 as the dose kernels would form it."""
    Dh = tf32_rn(D); Dl = tf32_rn(D - Dh); Th = tf32_rn(T); Tl = tf32_rn(T - Th)
    K, A = T.shape
    G = A // 32
    zero = lambda: np.zeros((K, D.shape[0]), np.float32)
    ks = [slice(g * 32 + j * 8, g * 32 + j * 8 + 8) for g in range(G) for j in range(4)]
    if layout in ("sep", "split2"):      # k_dose_tc: main accumulator(s) + separate correction accumulator
        mains, corr = [zero() for _ in range(1 if layout == "sep" else 2)], zero()
        for i, s in enumerate(ks):
            b = (i // 4) * len(mains) // G
            mains[b] = mma(mains[b], Th[:, s], Dh[:, s].T)
            corr = mma(corr, Tl[:, s], Dh[:, s].T)
            if i % 4 == 3:
                for s2 in ks[i - 3:i + 1]:
                    corr = mma(corr, Th[:, s2], Dl[:, s2].T)
        out = corr
        for m_ in mains:
            out = (out + m_).astype(np.float32)
        return out
    if layout == "corrections_first":    # k_dose_tc_pair: one accumulator, the small products first
        acc = zero()
        for s in ks:
            acc = mma(acc, Th[:, s], Dl[:, s].T)
        for s in ks:
            acc = mma(acc, Tl[:, s], Dh[:, s].T)
        for s in ks:
            acc = mma(acc, Th[:, s], Dh[:, s].T)
        return acc
    raise ValueError(layout)


def grad_model(D, Rh, segs, separate_corr):
    Dh = tf32_rn(D); Dl = tf32_rn(D - Dh)
    hi = tf32_trunc(Rh); lo = tf32_trunc((Rh - hi).astype(np.float32))
    K, N = Rh.shape
    n_slabs = N // 16
    G = np.zeros((K, D.shape[1]), np.float32)
    for sg in range(segs):
        main = np.zeros_like(G); corr = np.zeros_like(G)
        for p in range(sg * n_slabs // segs * 16, (sg + 1) * n_slabs // segs * 16, 8):
            s = slice(p, p + 8)
            main = mma(main, hi[:, s], Dh[s])
            if separate_corr:
                corr = mma(mma(corr, hi[:, s], Dl[s]), lo[:, s], Dh[s])
            else:
                main = mma(mma(main, hi[:, s], Dl[s]), lo[:, s], Dh[s])
        G = (G + (main + corr).astype(np.float32)).astype(np.float32)
    return G


def model_errors(n_cath, n_pos, layout, n_plans=24):
    """Threshold-sitting plans (the worst case of tests/test_gpu_parity.py) through the model; errors against the oracle."""
    c = gc.make_case("C1", n_cath=n_cath, n_pos=n_pos, counts=(700, 130, 250, 190), n_plans=n_plans, seed_points=9)
    T = np.repeat(c.T0[None], n_plans, axis=0) * np.linspace(0.85, 1.15, n_plans)[:, None].astype(np.float32)
    ref = oracle.evaluate(c.D, c.structures, T, c.weights)
    A, A_pad = c.n_dwell, (c.n_dwell + 31) // 32 * 32
    blocks, sid, valid, off = [], [], [], 0
    for si, s in enumerate(c.structures):                    # the library's row layout: structures padded to 64 rows
        n_pad = (s.n_points + 63) // 64 * 64
        blk = np.zeros((n_pad, A_pad), np.float32); blk[:s.n_points, :A] = c.D[off:off + s.n_points]
        blocks.append(blk); sid += [si] * n_pad; valid += [True] * s.n_points + [False] * (n_pad - s.n_points); off += s.n_points
    Dp, sid, valid = np.concatenate(blocks), np.array(sid), np.array(valid)
    x = np.zeros((n_plans, A_pad), np.float32); x[:, :A] = np.sqrt(T)
    d = dose_model(Dp, (x * x).astype(np.float32), layout)
    st = c.structures
    d_lo = np.array([st[s].d_lo for s in sid], np.float32); d_hi = np.array([st[s].d_hi for s in sid], np.float32)
    scale_lo = np.array([st[s].w_lo / st[s].n_points for s in sid], np.float32)
    scale_hi = np.array([st[s].w_hi / st[s].n_points for s in sid], np.float32)
    w = c.weights.astype(np.float32)
    W_lo = (w[:, sid, 0] * scale_lo[None]).astype(np.float32); W_hi = (w[:, sid, 1] * scale_hi[None]).astype(np.float32)
    Rh = ((W_lo * np.minimum(d - d_lo[None], np.float32(0))).astype(np.float32)
          + (W_hi * np.maximum(d - d_hi[None], np.float32(0))).astype(np.float32)).astype(np.float32)
    Rh[:, ~valid] = 0
    Gm = grad_model(Dp, Rh, min(74, Dp.shape[0] // 16), A_pad <= 256)
    g = (np.float32(4) * x * Gm).astype(np.float32)[:, :A]
    starts = np.cumsum([0] + [b.shape[0] for b in blocks[:-1]])
    dose = np.concatenate([d[:, o:o + s.n_points] for o, s in zip(starts, st)], axis=1).T
    e_d = float((np.abs(dose - ref["dose"]) / np.abs(ref["dose"])).max())
    e_g = float((np.linalg.norm(g - ref["grad_x"], axis=1) / np.linalg.norm(ref["grad_x"], axis=1)).max())
    return e_d, e_g


def test_model_of_the_layouts_in_use_and_of_the_candidate_for_wide_cases():
    # at 256 positions both layouts in use (separate correction accumulator / corrections first) behave alike
    d_sep, g_sep = model_errors(16, 16, "sep")
    d_cf, g_cf = model_errors(16, 16, "corrections_first")
    assert d_sep < 3e-6 and d_cf < 3e-6 and g_sep < 5e-5 and g_cf < 5e-5
    assert 0.7 < g_cf / g_sep < 1.4
    # at 384 positions the error grows with the number of adds into the main accumulator (48 instead of 32) ...
    d_w, g_w = model_errors(24, 16, "sep")
    assert d_w > d_sep and g_w > g_sep
    # ... and splitting the 48 adds over two accumulators (summed in fp32 registers by the epilogue) about halves it:
    # the designed fix for the XFAIL of test_gpu_parity.py, not applied without a GPU to validate it
    d_s2, g_s2 = model_errors(24, 16, "split2")
    assert g_s2 < 0.65 * g_w and d_s2 < 0.65 * d_w
    assert 2.4 * g_s2 < 1e-4             # with round 1's measured / model ratio the split layout would meet the bar
