"""CPU oracle for the SU(3)xSU(3) streaming hot path.  TEST INFRASTRUCTURE ONLY:
imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` legs; never by the product package."""
from .su3_oracle import (Geom, convert, convert_vec, cshift, index_vec, matvec, default_simd, expr, expr_real, index, mul_shift, neighbour, mul, mul3, mul_add, num_threads,
                         set_num_threads, site_to_outer, stream_triad)

__all__ = ["Geom", "convert", "convert_vec", "cshift", "index_vec", "matvec", "default_simd", "expr", "expr_real", "index", "mul_shift", "neighbour", "mul", "mul3", "mul_add", "num_threads",
           "set_num_threads", "site_to_outer", "stream_triad"]
