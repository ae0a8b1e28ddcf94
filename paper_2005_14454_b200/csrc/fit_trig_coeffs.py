import numpy as np
from numpy.polynomial import chebyshev as Ch
np.set_printoptions(precision=17)
ld = np.longdouble
def remez_like(fun, basis_pows, a, b, weight, iters=30, n=4000):
    # iteratively reweighted least squares approximating minimax of weight*(fun - poly)
    x = (np.cos(np.pi*(np.arange(n)+0.5)/n)*(b-a)/2 + (b+a)/2).astype(ld)
    A = np.stack([x**p for p in basis_pows], axis=1)
    y = fun(x)
    w = weight(x)
    wt = np.ones_like(x)
    for it in range(iters):
        W = (w*wt)[:,None]
        coef, *_ = np.linalg.lstsq((A*W).astype(np.float64), (y*w*wt).astype(np.float64), rcond=None)
        err = np.abs((A@coef.astype(ld) - y)*w)
        wt = wt*(1 + 5*(err/err.max())**2); wt/=wt.mean()
    return coef, float(err.max())
# sin(r) - r = r^3 P(r^2): basis r^3,r^5,r^7,r^9 ; weight 1/|r| (relative)
a=1e-6; b=np.pi/4*1.0001
cs, es = remez_like(lambda x: np.sin(x)-x, [3,5,7,9], a, b, lambda x: 1/np.abs(x))
print("sin coefs", [repr(float(np.float32(c))) for c in cs], es)
cs3, es3 = remez_like(lambda x: np.sin(x)-x, [3,5,7], a, b, lambda x: 1/np.abs(x))
print("sin coefs deg7", [repr(float(np.float32(c))) for c in cs3], es3)
cc, ec = remez_like(lambda x: np.cos(x)-1+x*x/2, [4,6,8], a, b, lambda x: 1+0*x)
print("cos coefs", [repr(float(np.float32(c))) for c in cc], ec)
c1=np.float32(np.pi/2); c2=np.float32(np.pi/2-np.float64(c1)); c3=np.float32(np.pi/2-np.float64(c1)-np.float64(c2))
print(repr(float(c1)), repr(float(c2)), repr(float(c3)), repr(float(np.float32(2/np.pi))))
b2=np.pi/2*1.0001
for pows in ([3,5,7,9],[3,5,7,9,11]):
    c, e = remez_like(lambda x: np.sin(x)-x, pows, a, b2, lambda x: 1/np.abs(x))
    print("sin halfpi", pows, [repr(float(np.float32(v))) for v in c], e)
c1=np.float32(np.pi); c2=np.float32(np.pi-np.float64(c1)); 
print(repr(float(c1)), repr(float(c2)), repr(float(np.float32(1/np.pi))))
