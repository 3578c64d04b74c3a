"""Concrete seeded inputs for BASELINE.json configs (recipe: DESIGN.md "Input recipe")."""
from __future__ import annotations

import numpy as np

from .chirps import ChirpParams, draw_chirp_params, inject_chirps
from .noise import coloured_noise

FS = 2048


def config0_strain():
    """configs[0]: 2 channels, 64 s of coloured noise, seed 1000."""
    return coloured_noise(64 * FS, seed=1000)


def config1_raw(n_windows=128, kernel_len=3072, seed=1001):
    """configs[1]: raw strain holding n_windows/2 chirps (SNR U(4,20)), and the raw-sample index at which
    each of the n_windows windows starts: chirp windows (coalescence time uniform in [0.25, 1.25] s of
    the window) interleaved with noise-only windows taken >= 6 s from any chirp."""
    n_ch = n_windows // 2
    rng = np.random.Generator(np.random.PCG64(seed + 7))
    t_first = 70.0
    dur = int(t_first + 2.0 * n_ch + 8.0)
    noise = coloured_noise(dur * FS, seed=seed)
    params, starts_chirp = [], []
    for i in range(n_ch):
        t_c = t_first + 2.0 * i + rng.uniform(0.0, 0.5)
        params.append(ChirpParams(t_c=float(t_c), m_chirp=float(rng.uniform(10, 60)), phi0=float(rng.uniform(0, 2 * np.pi)),
                                  delta_l1=float(rng.uniform(-0.01, 0.01)), snr=float(rng.uniform(4, 20))))
        starts_chirp.append(int(round((t_c - rng.uniform(0.25, 1.25)) * FS)))
    strain, _ = inject_chirps(noise, params)
    starts_noise = [int((4.0 + 0.75 * i) * FS) for i in range(n_windows - n_ch)]
    assert starts_noise[-1] + kernel_len < (t_first - 6.0 - 5.0) * FS
    starts = []
    for i in range(n_windows):
        starts.append(starts_chirp[i // 2] if i % 2 == 0 and i // 2 < n_ch else starts_noise[i // 2])
    return strain, np.asarray(starts, dtype=np.int64), params


def gather_windows(white, starts, kernel_len, offset):
    """windows[i][c] = white[c][starts[i] - offset : ... + kernel_len]; offset = raw index of white[:, 0]."""
    return np.stack([white[:, s - offset: s - offset + kernel_len] for s in starts])


def config2_strain(duration_s=3600, n_chirps=200, seed=1002):
    """configs[2] (also fed update by update as configs[4]): `duration_s` of two-detector coloured noise (seed 1002) with
    one Newtonian chirp per 17.6 s slot from t = 70 s on (200 in the hour), chirp mass U(10, 60) Msun, per-detector
    offset U(+-10 ms), network SNR U(4, 20).  Returns (strain float32 [2][N], chirp parameters)."""
    noise = coloured_noise(int(duration_s) * FS, seed=seed)
    params = draw_chirp_params(n_chirps, float(duration_s), seed=seed + 7)
    strain, _ = inject_chirps(noise, params)
    return strain, params


def config3_block(index, n_raw):
    """One time block of the configs[3] record (1e5 s analysed in independent blocks): coloured noise with its own seed
    and chirps at configs[2]'s rate and parameter ranges (one per 17.6 s slot after the 64 s PSD history)."""
    seed = int(np.random.SeedSequence([1003, int(index)]).generate_state(1)[0])
    noise = coloured_noise(int(n_raw), seed=seed)
    dur = n_raw / FS
    params = draw_chirp_params(int(dur // 17.6) + 1, dur, seed=seed + 7)
    strain, _ = inject_chirps(noise, params)
    return strain, params
