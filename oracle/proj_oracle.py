"""Plain definition of the two projections either side of the attention -- TEST INFRASTRUCTURE, not the product.

Only tests/ may import this.  float64 numpy, one einsum per projection (a library contraction as the single step), written
from the definition in include/kairos.h / SURVEY.md 8(c) (absorbed MLA of the model the paper serves):

  absorb_q     q[j,h,0:512]   = sum_k q_nope[j,h,k] * W_UK[h,d,k]      q[j,h,512:576] = q_rope[j,h,:]
  project_out  v[j,h,e]       = sum_d o_lat[j,h,d]  * W_UV[h,e,d]

Inputs are bf16 bit patterns (uint16) or float arrays; outputs are UNROUNDED float64 (the GPU's bf16 results are compared
within a tolerance).  Pinned in tests/test_proj.py by identity / one-hot weights worked by hand and by the identity
"absorbed attention followed by W_UV == ordinary multi-head attention with k = [W_UK c | kR], v = W_UV c" against a dense
softmax written out separately.  Shares no code with csrc/proj.cu.
"""
from __future__ import annotations

import numpy as np

from paper_2607_02043_b200 import workloads as W


def _f64(x: np.ndarray) -> np.ndarray:
    return W.bf16_bits_to_f32(x).astype(np.float64) if x.dtype == np.uint16 else np.asarray(x, dtype=np.float64)


def absorb_q(q_nope, q_rope, w_uk_t) -> np.ndarray:
    """q_nope [n,16,128], q_rope [n,16,64], w_uk_t [16,512,128] -> q [n,16,576] (float64)."""
    qn, qr, w = _f64(q_nope), _f64(q_rope), _f64(w_uk_t)
    lat = np.einsum("jhk,hdk->jhd", qn, w)
    return np.concatenate([lat, qr], axis=2)


def project_out(o_lat, w_uv_t) -> np.ndarray:
    """o_lat [n,16,512], w_uv_t [16,128,512] -> v [n,16,128] (float64)."""
    return np.einsum("jhd,hed->jhe", _f64(o_lat), _f64(w_uv_t))
