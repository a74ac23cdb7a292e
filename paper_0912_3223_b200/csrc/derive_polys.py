"""derive_polys.py — where the polynomial coefficients in lpm_device.cuh come from.

    python paper_0912_3223_b200/csrc/derive_polys.py

Own minimax-style fits (Lawson-weighted least squares on Chebyshev nodes) for the three elementary
functions of the Box-Muller step (R3), on exactly the argument ranges that can occur:
  log1p(f) = f + f^2 P(f),            f in [-1/3, 1/3]      (degree 7: the CLOG line)
  sin(pi r) = r (pi + r^2 S(r^2)),    r in [-1/4, 1/4]      (degree 2 in r^2: CSIN)
  cos(pi r) = 1 + r^2 C(r^2),         r in [-1/4, 1/4]      (degree 3 in r^2: CCOS)
Prints the fp32-rounded coefficients and the fit errors in exact arithmetic; the fp32 evaluation error
is checked exhaustively on the GPU over all 2^24 arguments (tests/test_gpu_parity.py::
test_box_muller_exhaustive).  This script belongs to the CUDA path only: the oracle calls libm in fp64.
"""
import numpy as np
from numpy.polynomial import chebyshev as Ch, polynomial as P
np.set_printoptions(precision=17)
f32=np.float32
def fma(a,b,c): return (a.astype(np.float64)*b.astype(np.float64)+np.float64(c)).astype(f32)

def cheb_fit(fun, lo, hi, deg, n=4000, w=None):
    # least squares at Chebyshev nodes ~ near-minimax
    k=np.arange(n); x=np.cos(np.pi*(k+0.5)/n); t=0.5*(hi-lo)*x+0.5*(hi+lo)
    y=fun(t)
    c=P.polyfit(t,y,deg,w=w(t) if w else None)
    return c

def remez_like(fun, lo, hi, deg, iters=30, wfun=None):
    # iteratively reweighted LSQ (Lawson) for minimax of relative/abs error
    n=6000; k=np.arange(n); x=np.cos(np.pi*(k+0.5)/n); t=0.5*(hi-lo)*x+0.5*(hi+lo)
    y=fun(t); w=np.ones(n)
    base = wfun(t) if wfun else np.ones(n)
    for _ in range(iters):
        c=P.polyfit(t,y,deg,w=np.sqrt(w)*base)
        e=np.abs(P.polyval(t,c)-y)*base
        w=w*(e/e.max()+1e-3); w/=w.sum()
    return c

# ---- log1p(f) = f + f*f*P1(f), f in [-1/3, 1/3]
def g(f):
    f=np.where(f==0,1e-300,f)
    return (np.log1p(f)-f)/(f*f)
for deg in (7,8,9):
    c=remez_like(g,-1/3,1/3+1e-9,deg)
    t=np.linspace(-1/3,1/3,200001); t=t[t!=0]
    approx=t+t*t*P.polyval(t,c)
    print("log deg",deg,"max rel err",np.max(np.abs(approx/np.log1p(t)-1)))
    if deg==8: clog=c
print("clog",[float(f32(v)) for v in clog])

# ---- sin(pi r)= r*(pi + r2*S(r2)); cos(pi r)=1+r2*C(r2), r in [-1/4,1/4], s=r2 in [0,1/16]
def gs(s):
    r=np.sqrt(np.maximum(s,1e-300)); return (np.sin(np.pi*r)/r-np.pi)/s
def gc(s):
    r=np.sqrt(np.maximum(s,1e-300)); return (np.cos(np.pi*r)-1)/s
for deg in (2,3,4):
    cs=remez_like(gs,1e-12,1/16,deg); cc=remez_like(gc,1e-12,1/16,deg)
    r=np.linspace(-0.25,0.25,200001); s=r*r
    es=np.max(np.abs(r*(np.pi+s*P.polyval(s,cs))-np.sin(np.pi*r)))
    ec=np.max(np.abs(1+s*P.polyval(s,cc)-np.cos(np.pi*r)))
    print("sincos deg",deg,es,ec)
    if deg==3: csin,ccos=cs,cc
print("csin",[float(f32(v)) for v in csin]); print("ccos",[float(f32(v)) for v in ccos])
if __name__ == "__main__":
    f32 = np.float32
    print("CLOG", [repr(float(f32(v))) for v in remez_like(g, -1/3, 1/3 + 1e-9, 7)])
    print("CSIN", [repr(float(f32(v))) for v in remez_like(gs, 1e-12, 1/16, 2)])
    print("CCOS", [repr(float(f32(v))) for v in remez_like(gc, 1e-12, 1/16, 3)])
