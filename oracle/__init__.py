"""Float64 CPU oracle of the LLOID hot path -- test infrastructure only (see lloid_oracle.py header)."""
from .lloid_oracle import (  # noqa: F401
    N_DOWN, N_UP, Series, resample_kernel, decimate, upsample, upsample_input_range,
    basis_correlate, reconstruct, rate_groups, lloid_snr, brute_force, find_peaks,
)
from .events_oracle import find_peaks_overlap, template_acorr, xi2, coincidences, cluster  # noqa: F401,E402
from .whiten_oracle import Whitener, log_median_mean, hann_periodic, tukey_taper  # noqa: F401,E402
from .svd_oracle import svd_slice  # noqa: F401,E402
