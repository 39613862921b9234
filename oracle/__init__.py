"""CPU oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT) -- see fe_oracle.h.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package; the CUDA product (paper_2510_10529_b200/) never does, and this package never imports the product.
"""
from .fe_oracle import (  # noqa: F401
    OracleMesh, build_oracle, gll, gauss, lagrange, lagrange_deriv, lanczos_bounds, rayleigh_ritz,
    laplacian_precond, minres_shifted, density, adjoint_rhs, ritz_residuals, chfsi,
)
from .fe_general import GeneralOracleMesh  # noqa: F401,E402
