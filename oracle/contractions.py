"""O2. Elementary local contractions (oracle, test infra).

Index convention (BASELINE.json north_star): environments L[a, w, x] and R[b, v, y] carry the
bra (conjugated) bond index first and the ket bond index last; W[w, s, t, v] has s = bra (output)
and t = ket (input) physical index; site tensors A[x, t, y].

  heff  : Eq. 29 applied to a site tensor as in Eq. 43
  envL/R: Eq. 30-32, one more site absorbed into h[1:i] / h[i:N]
  bond  : Eq. 44

Each operation is given twice: ``*_definition`` is the defining sum as ONE einsum (slow: numpy
evaluates it without BLAS); the working version contracts "small matrices one by one"
 with numpy.tensordot, one library matmul per tensor, in the order L, W, R.  The
two are compared in tests/test_oracle_pins.py.
"""
import numpy as np


def heff_definition(L, W, A, R):
    """out[a,s,b] = sum L[a,w,x] W[w,s,t,v] A[x,t,y] R[b,v,y]."""
    return np.einsum("awx,wstv,xty,bvy->asb", L, W, A, R)


def envL_definition(L, W, A):
    """L'[b,v,y] = sum conj(A[a,s,b]) L[a,w,x] W[w,s,t,v] A[x,t,y]."""
    return np.einsum("asb,awx,wstv,xty->bvy", A.conj(), L, W, A)


def envR_definition(R, W, A):
    """R'[a,w,x] = sum conj(A[a,s,b]) W[w,s,t,v] A[x,t,y] R[b,v,y]."""
    return np.einsum("asb,wstv,xty,bvy->awx", A.conj(), W, A, R)


def bond_definition(L, D, R):
    """D'[a,b] = sum L[a,w,x] D[x,y] R[b,w,y]."""
    return np.einsum("awx,xy,bwy->ab", L, D, R)


def heff(L, W, A, R):
    T1 = np.tensordot(L, A, axes=([2], [0]))               # [a,w,t,y]
    T2 = np.tensordot(T1, W, axes=([1, 2], [0, 2]))        # [a,y,s,v]
    return np.tensordot(T2, R, axes=([3, 1], [1, 2]))      # [a,s,b]


def envL(L, W, A):
    T1 = np.tensordot(L, A, axes=([2], [0]))               # [a,w,t,y]
    T2 = np.tensordot(T1, W, axes=([1, 2], [0, 2]))        # [a,y,s,v]
    out = np.tensordot(A.conj(), T2, axes=([0, 1], [0, 2]))  # [b,y,v]
    return np.ascontiguousarray(out.transpose(0, 2, 1))    # [b,v,y]


def envR(R, W, A):
    T1 = np.tensordot(A, R, axes=([2], [2]))               # [x,t,b,v]
    T2 = np.tensordot(W, T1, axes=([2, 3], [1, 3]))        # [w,s,x,b]
    return np.tensordot(A.conj(), T2, axes=([1, 2], [1, 3]))  # [a,w,x]


def bond(L, D, R):
    T = np.tensordot(L, D, axes=([2], [0]))                # [a,w,y]
    return np.tensordot(T, R, axes=([1, 2], [1, 2]))       # [a,b]


def boundary_env():
    """h[1:0] = h[N+1:N] = 1 (Eq. 23)."""
    return np.ones((1, 1, 1), dtype=np.complex128)
