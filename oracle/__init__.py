"""CPU oracle for the MSM hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package. It never imports paper_2510_05961_b200's CUDA binding.
"""
from .oracle import Oracle, build, lib, gamma, dgamma, kernel, dkernel, bspline, dbspline, \
    two_scale, omega, direct_sum

__all__ = ["Oracle", "build", "lib", "gamma", "dgamma", "kernel", "dkernel", "bspline",
           "dbspline", "two_scale", "omega", "direct_sum"]
