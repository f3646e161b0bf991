"""Acceptance checks GPU-vs-oracle (BASELINE.json north_star; DESIGN.md §5 'Tolerances')."""
import numpy as np

FEATURE_ATOL = 1e-3          # "encoded features within 1e-3 absolute (fp16 texels, fp32 accumulate)"
RGB_MAX_ABS = 2e-2           # "final RGB within max-abs 2e-2 ..."
RGB_MEAN_ABS = 2e-3          # "... and mean-abs 2e-3 on outputs in [0,4]"
RGB_REL_ABOVE_4 = 5e-3       # A23: above 4 the same bound relatively (2e-2 / 4)
# d^ = exp(z) of the disparity predictor: the GPU rounds the network input and both hidden activations to
# fp16 (2^-11 relative each); with He-normal weights and O(1) activations that perturbs z by about
# sqrt(64) * 0.18 * 2^-11 * sqrt(3) ~ 1.2e-3 (random signs), a few times that at the maximum over 1e4-1e5 queries, and
# |delta d^| / d^ = |delta z|.  north_star states no bound for this output; 5e-3 (the relative form of its RGB bound, A23) is ~6x the 8.4e-4 measured
# on B200 over 20,037 queries.
DISPARITY_REL = 5e-3


def check_indices(slot_gpu, tex_gpu, slot_ref, tex_ref):
    assert np.array_equal(np.asarray(slot_gpu, np.int64), np.asarray(slot_ref, np.int64)), "node/slot indices differ"
    assert np.array_equal(np.asarray(tex_gpu, np.int64), np.asarray(tex_ref, np.int64)), "texel indices differ"


def check_features(f_gpu, f_ref, storage="f16"):
    f_gpu = np.asarray(f_gpu, np.float64)
    err = np.abs(f_gpu - f_ref)
    # the stored feature is rounded once to the tree dtype: fp16 spacing is 2^-11 relative, well inside 1e-3 for |h| < 1
    assert err.max() <= FEATURE_ATOL, "feature max-abs error %.3g > %.3g" % (err.max(), FEATURE_ATOL)
    return float(err.max())


def check_rgb(rgb_gpu, rgb_ref):
    rgb_gpu = np.asarray(rgb_gpu, np.float64)
    assert np.isfinite(rgb_gpu).all()
    err = np.abs(rgb_gpu - rgb_ref)
    low = rgb_ref <= 4.0
    if low.any():
        assert err[low].max() <= RGB_MAX_ABS, "rgb max-abs error %.3g > %.3g" % (err[low].max(), RGB_MAX_ABS)
        assert err[low].mean() <= RGB_MEAN_ABS, "rgb mean-abs error %.3g > %.3g" % (err[low].mean(), RGB_MEAN_ABS)
    if (~low).any():
        rel = err[~low] / rgb_ref[~low]
        assert rel.max() <= RGB_REL_ABOVE_4, "rgb relative error above 4: %.3g > %.3g" % (rel.max(), RGB_REL_ABOVE_4)
    return float(err[low].max()) if low.any() else 0.0, float(err[low].mean()) if low.any() else 0.0
