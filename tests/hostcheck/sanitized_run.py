"""Runs the oracle and the host-compiled per-element math of the CUDA path, both built with -fsanitize=address,undefined, over seeded
stress inputs (started by tests/test_sanitizers.py with the sanitizer runtimes preloaded).  argv: sanitized liboracle, sanitized libhostcheck."""
import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from paper_2212_01937_b200 import workloads as W
DP = C.POINTER(C.c_double); LDP = C.POINTER(C.c_longdouble)
orc = C.CDLL(sys.argv[1]); hc = C.CDLL(sys.argv[2])
w = W.config5(n=1500, n_struct=300)
n = w.n_z
dp = lambda a: np.ascontiguousarray(a, dtype=np.float64).ctypes.data_as(DP)
val = np.zeros((n, 6), dtype=np.longdouble); grad = np.zeros((n, 6, 5), dtype=np.longdouble); st = np.zeros(n, dtype=np.int32)
orc.oracle_observables_batch.argtypes = [C.c_int64, DP, DP, DP, DP, DP, C.c_int64, LDP, LDP, C.POINTER(C.c_int32)]
orc.oracle_observables_batch(n, dp(w.z), dp(w.Om), dp(w.OL), dp(w.Or), dp(w.H0), n, val.ctypes.data_as(LDP), grad.ctypes.data_as(LDP), st.ctypes.data_as(C.POINTER(C.c_int32)))
wm = W.wmix(n=800); m = len(wm["z"])
v6 = np.zeros((m, 6), dtype=np.longdouble); g6 = np.zeros((m, 6, 7), dtype=np.longdouble); s6 = np.zeros(m, dtype=np.int32)
orc.oracle_w_observables_batch.argtypes = [C.c_int64] + [DP] * 7 + [C.c_int64, LDP, LDP, C.POINTER(C.c_int32)]
orc.oracle_w_observables_batch(m, *[dp(wm[k]) for k in ("z", "Om", "OL", "Or", "Ow13", "Ow23", "H0")], m, v6.ctypes.data_as(LDP), g6.ctypes.data_as(LDP), s6.ctypes.data_as(C.POINTER(C.c_int32)))
out = np.zeros((9, n)); gz = np.zeros(n); gp = np.zeros((4, n)); sb = np.zeros(n, dtype=np.uint8)
gup = np.random.default_rng(0).standard_normal((9, n))
for f in (hc.hostcheck_f64, hc.hostcheck_elem_f64, hc.hostcheck_elem_f32):
    f(C.c_int64(n), dp(w.z), dp(w.Om), dp(w.OL), dp(w.Or), dp(w.H0), C.c_uint(511), dp(gup), dp(out), dp(gz), dp(gp), sb.ctypes.data_as(C.POINTER(C.c_uint8)))
vw = np.zeros((6, m)); dw = np.zeros((6, m)); gw = np.zeros((6, 6, m)); sw = np.zeros(m, dtype=np.uint8)
hc.hostcheck_w_full(C.c_int64(m), *[dp(wm[k]) for k in ("z", "Om", "OL", "Or", "Ow13", "Ow23", "H0")], dp(vw), dp(dw), dp(gw), sw.ctypes.data_as(C.POINTER(C.c_uint8)))
z1 = np.random.default_rng(1).uniform(0, 3, 500); z2 = z1 + 0.5
t5 = np.zeros((5, 500)); t1 = np.zeros((5, 500)); t2 = np.zeros((5, 500)); tp = np.zeros((5, 4, 500)); ts = np.zeros(500, dtype=np.uint8)
hc.hostcheck_two(C.c_int64(500), dp(z1), dp(z2), dp(w.Om[:500]), dp(w.OL[:500]), dp(w.Or[:500]), dp(w.H0[:500]), dp(t5), dp(t1), dp(t2), dp(tp), ts.ctypes.data_as(C.POINTER(C.c_uint8)))
print("sanitized run finished: oracle (LCDM + w family), host-compiled CUDA math (OUTER, ELEMENTWISE f64/f32 sequences, w family, two-limit)")
