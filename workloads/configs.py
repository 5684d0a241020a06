"""The five workload configurations of BASELINE.json, as plain data.

Derived counts follow SURVEY.md §8 "Sizes per config".  Sub-streams of the
seed are spawned in the fixed order *bank, strain, sky, injections, snippets*
(SURVEY.md §8(d)); base seed = 20110678 + config index.
"""
import numpy as np

BASE_SEED = 20110678

RATES8 = [4096, 2048, 1024, 512, 256, 128, 64, 32]

CONFIGS = {
    0: dict(name="cfg0-tiny", dets=["H1", "L1"], sigma=[1.0, 1.0], seconds=1,
            band_rates=[2048], out_band=0, n_templates=4, filters_per_template=32,
            nside=4, threshold=0.0, n_slides=0, n_chirp_templates=0, injections=0),
    1: dict(name="cfg1-hlv-512x300", dets=["H1", "L1", "V1"], sigma=[1.0, 1.0, 0.5], seconds=16,
            band_rates=[2048], out_band=0, n_templates=512, filters_per_template=300,
            nside=16, threshold=4.0, n_slides=0, n_chirp_templates=1, injections=1,
            chirp=dict(f0=30.0, tc=12.0, t_start=2.0, snr=15.0)),
    2: dict(name="cfg2-multirate-1024x600", dets=["H1", "L1"], sigma=[1.0, 1.0], seconds=64,
            band_rates=RATES8, out_band=1, n_templates=1024, filters_per_template=600,
            nside=0, threshold=4.0, n_slides=0, n_chirp_templates=0, injections=0),
    3: dict(name="cfg3-sky-stress", dets=["H1", "L1", "V1"], sigma=[1.0, 1.0, 0.5], seconds=1,
            band_rates=[2048], out_band=0, n_templates=0, filters_per_template=0,
            nside=64, threshold=4.0, n_slides=100, n_triggers=4096, snippet_half=102,
            coherent_fraction=0.10, n_chirp_templates=0, injections=0),
    4: dict(name="cfg4-full-20000x700", dets=["H1", "L1", "V1"], sigma=[1.0, 1.0, 0.5], seconds=128,
            band_rates=RATES8, out_band=1, n_templates=20000, filters_per_template=700,
            nside=32, threshold=4.0, n_slides=100, n_chirp_templates=20, injections=20),
}


def config(idx):
    c = dict(CONFIGS[idx])
    c["index"] = idx
    c["seed"] = BASE_SEED + idx
    c["f_out"] = 2048
    return c


def streams(seed):
    """Five independent numpy Generators: bank, strain, sky, injections, snippets."""
    ss = np.random.SeedSequence(seed).spawn(5)
    names = ["bank", "strain", "sky", "injections", "snippets"]
    return {n: np.random.Generator(np.random.PCG64(s)) for n, s in zip(names, ss)}
