"""NEXT-1  post-processing of the score series.  (Oracle: test infrastructure only.)

Paper: "These neural-network predictions are then integrated over time using a 1 s top hat filter (see Fig. 1) [...]
Finally, the integrated timeseries of neural-network predictions is clustered to avoid yielding multiple triggers for
the same event.  The maximum integrated value over an 8 s window is taken as the detection statistic corresponding to
a candidate event." (Sec. II; latency rows "Integrating network output" / "Identifying candidate events",
P:209.)

The paper fixes the durations only.  Readings (D1-D3):
  D1  top hat = the MEAN of the trailing n_int = rate * 1 s scores (causal: entry i covers scores i - n_int + 1 .. i);
      the first n_int - 1 entries average the scores that exist (a monotone rescaling of a sum; ranks are unaffected).
  D2  clustering = consecutive, non-overlapping windows of n_cluster = rate * 8 s integrated values; each yields one
      trigger (index of the FIRST maximum, its value); a trailing partial window yields one too.
  D3  the integer decision (argmax) is taken in the kernel's precision: float32 sums in index order, then one multiply.
"""
from __future__ import annotations

import numpy as np


def integrate_tophat(scores, n_int, dtype=np.float64):
    """I[i] = (1/m) sum_{j=max(0,i-n_int+1)}^{i} s[j], m = number of terms, summed in index order in `dtype`."""
    s = np.asarray(scores, dtype=dtype)
    out = np.empty_like(s)
    for i in range(s.shape[0]):
        lo = max(0, i - n_int + 1)
        acc = dtype(0)
        for j in range(lo, i + 1):
            acc = dtype(acc + s[j])
        out[i] = dtype(acc * dtype(dtype(1) / dtype(i + 1 - lo)))
    return out


def cluster_max(integrated, n_cluster):
    """Per consecutive window of n_cluster values: (index of the first maximum, maximum)."""
    x = np.asarray(integrated)
    idx, val = [], []
    for a in range(0, x.shape[0], n_cluster):
        w = x[a: a + n_cluster]
        k = int(np.argmax(w))            # numpy returns the first maximum
        idx.append(a + k)
        val.append(w[k])
    return np.asarray(idx, dtype=np.int64), np.asarray(val, dtype=x.dtype)
