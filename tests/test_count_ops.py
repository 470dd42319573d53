"""The op-counting build of the oracle (oracle/opcount.h, oracle/count_ops.py) compiles, computes the same
numbers as the plain build and counts what can be counted by hand."""
import ctypes as C
import os

import numpy as np


def test_counting_build_counts_and_computes_the_same(orc):
    from oracle import count_ops
    so = count_ops.build()
    L = C.CDLL(so)
    vp = C.c_void_p
    L.tfo_flux_maxwell.argtypes = [vp, vp, vp, C.c_double, C.c_double, vp]
    L.tfo_opcount_get.argtypes = [C.POINTER(C.c_int64)]
    ph = orc.physics_c()
    rng = np.random.default_rng(0)
    UL, UR = rng.normal(size=8), rng.normal(size=8)
    H = np.empty(8)
    L.tfo_opcount_reset()
    L.tfo_flux_maxwell(C.byref(ph), UL.ctypes.data_as(vp), UR.ctypes.data_as(vp), 0.6, 0.8, H.ctypes.data_as(vp))
    cnt = (C.c_int64 * 8)()
    L.tfo_opcount_get(cnt)
    np.testing.assert_array_equal(H, orc.flux_maxwell(ph, UL, UR, 0.6, 0.8))       # same arithmetic, same bits
    # by hand from oracle/tfo.cpp: H = 1/2 (H_L + H_R) - 1/2 alpha D per row is 2 additions and 3 multiplications
    # (8 rows), U_R - U_L 8 subtractions; the rest sits in the two physical fluxes and in |A_n| dU
    add, mul, div, sqrt = cnt[0], cnt[1], cnt[2], cnt[3]
    assert div == 0 and sqrt == 0 and add >= 8 * 2 + 8 and mul >= 8 * 3
    assert (add, mul) == (54, 120)                                                  # the figures of profiles/r2_oracle_flops.md
    assert os.path.basename(so) == "liboracle_tfo_count.so"
