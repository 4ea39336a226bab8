"""CPU oracle of the XC quadrature (arxiv 2007.03143).  TEST INFRASTRUCTURE ONLY: imported by tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs -- never by the product
package.  See xc_oracle.cpp for the arithmetic and its citations."""
from .xc_oracle import *  # noqa: F401,F403
