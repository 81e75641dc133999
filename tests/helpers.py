"""Small model configurations shared by the oracle pins and the GPU parity tests."""
from paper_2512_24840_b200 import synth


def small_config(**kw):
    """A small single-segment log-grid model (592 px, K=10, D=4)."""
    base = dict(cfg=7, name="pin-small", B=4, grid="log10", lam_min=4800.0, lam_max=5500.0, step=1e-4,
                seg_bounds=None, sigma_inst=(0.0,), K=10, L=3, D=4, n_iter=50, snr=(50.0, 50.0),
                noise="const", mask_frac=0.03, parity_B=4)
    base.update(kw)
    return synth.Config(**base)


def two_arm_config(**kw):
    """Two segments on a LINEAR grid with instrumental widths (exercises C.2-13, -14)."""
    base = dict(cfg=8, name="pin-2arm", B=3, grid="linear", lam_min=5000.0, lam_max=5000.0 + 0.8 * 699,
                step=0.8, seg_bounds=(0, 380, 700), sigma_inst=(70.0, 45.0), K=10, L=3, D=3, n_iter=20,
                snr=(80.0, 80.0), noise="poisson", mask_frac=0.05, parity_B=3)
    base.update(kw)
    return synth.Config(**base)


def two_arm_log_config(**kw):
    """Two segments on a LOG grid with different instrumental widths (uniform kernels, several segments)."""
    base = dict(cfg=9, name="pin-2arm-log", B=5, grid="log10", lam_min=4500.0, lam_max=5600.0, step=1e-4,
                seg_bounds=(0, 500, 950), sigma_inst=(30.0, 60.0), K=12, L=3, D=6, n_iter=40, snr=(60.0, 60.0),
                noise="const", mask_frac=0.04, parity_B=5)
    base.update(kw)
    return synth.Config(**base)


def make(cfgobj, oracle_mod, B=None, noise_free=False):
    synth.CONFIGS["_tmp"] = cfgobj
    try:
        return synth.make_case("_tmp", oracle_mod.forward, B=B, noise_free=noise_free)
    finally:
        del synth.CONFIGS["_tmp"]
