"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds NONE of the method's arithmetic (no Welch, no filter design,
no whitening, no convolution, no norm fold).  It only produces inputs:

* ``noise``   -- coloured Gaussian strain standing in for GWOSC O3 data
                 (Sec. IV.A; recipe in SURVEY.md 8(d) / DESIGN.md).
* ``chirps``  -- analytic Newtonian chirps standing in for the paper's
                 IMRPhenomPv2 injections.
* ``weights`` -- seeded He-normal network parameters and the weight-blob
                 writer (the blob stores UNFOLDED parameters; each side folds
                 the norm itself).
"""
from .noise import analytic_psd, coloured_noise, SIGMA_X_ANALYTIC  # noqa: F401
from .chirps import newtonian_chirp, inject_chirps, ChirpParams  # noqa: F401
from .weights import (  # noqa: F401
    LayerSpec, resnet_layer_table, make_weight_blob, tiny_config, full_config, tiny_config_live_gn, full_config_live_gn,
    KIND_CONV, KIND_MAXPOOL, KIND_HEAD, NORM_CHANNEL, NORM_GROUP, NORM_GROUP_LIVE,
)
