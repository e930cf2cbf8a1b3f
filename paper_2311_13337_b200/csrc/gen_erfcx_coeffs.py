"""Generator of the FP32 erfcx approximation used by csrc/tvbx_tf.cuh (half_erfc<float>).

erfcx(a) = exp(a^2) erfc(a) for a >= 0 is written t * R(t) with t = 1 / (1 + p a); R is a polynomial
fitted here by weighted least squares (relative error) at Chebyshev nodes of t in (0, 1] against a
40-digit mpmath reference.  The script prints the maximum relative error of the approximation when
it is EVALUATED IN FP32 (Horner, as the kernel does) over a >= 0, then the coefficients of the chosen
(p, degree) in ascending powers of t.  Not used at run time; kept as the provenance of the constants.
"""
import mpmath as mp
import numpy as np
from scipy import special
mp.mp.dps=40
def ref(z): return float(mp.erfc(z)*mp.exp(mp.mpf(z)**2))
def fit(p,deg,npts=4000):
    # t in (0,1], z = (1/t - 1)/p
    k=np.arange(npts); t=0.5*(1-np.cos(np.pi*(k+0.5)/npts)); t=t*(1-1e-9)+1e-9
    z=(1/t-1)/p
    y=np.array([ref(zz) for zz in z])/t
    # weighted LS on relative error via Chebyshev basis on [0,1]
    x=2*t-1
    V=np.polynomial.chebyshev.chebvander(x,deg)
    A=V/y[:,None]
    c,*_=np.linalg.lstsq(A,np.ones_like(y),rcond=None)
    poly=np.polynomial.chebyshev.Chebyshev(c,domain=[0,1]).convert(kind=np.polynomial.Polynomial,domain=[0,1],window=[0,1])
    coef=poly.coef
    return coef
def test(coef,p):
    c32=coef.astype(np.float32)
    z=np.concatenate([np.linspace(0,12,200001),np.logspace(-6,2,20000)]).astype(np.float32)
    t=(np.float32(1)/(np.float32(1)+np.float32(p)*z)).astype(np.float32)
    r=np.zeros_like(t)+c32[-1]
    for c in c32[-2::-1]: r=(r*t+c).astype(np.float32)
    val=(r*t).astype(np.float64)
    refv=special.erfcx(z.astype(np.float64))
    rel=np.abs(val/refv-1)
    return rel.max()
for p in (0.5,0.7,1.0,0.4,0.3):
    for deg in (8,9,10,11,12):
        coef=fit(p,deg,1500)
        print(p,deg,test(coef,p))
print("----")
coef=fit(0.4,8,4000)
print(test(coef,0.4))
print(", ".join(f"{c:.9e}f" for c in coef))
