"""CPU oracle for the dfrg loop integrals -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It compiles oracle/dfrg_oracle.cpp with g++ (plain C++,
OpenMP across outputs) and exposes it through ctypes on numpy arrays.  It imports
nothing from paper_2412_13043_b200 and the CUDA path imports nothing from here.
"""
from .binding import (  # noqa: F401
    build,
    gl_rule,
    regulator,
    regulator_fermion,
    table_lookup,
    lpa,
    lpa_fermion,
    loop4d_twopoint,
    loop4d_threepoint,
    loop4d_fourpoint,
    loop4d_threepoint_tab3d,
    table3d_lookup,
    vertex_coords,
    matsubara3d,
    matsubara3d_mu,
    matsubara3d_mu_dm2,
    lpa_dm2,
    loop4d_twopoint_dm2,
    matsubara3d_dm2,
    num_threads,
    set_num_threads,
    REG_LITIM,
    REG_EXP_POLY,
)
