"""CPU oracle of the batch RGBD rasteriser -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It imports nothing from paper_2306_07552_b200 and shares no code with the CUDA path.
"""
from .gx_oracle import (build, render, raster_soup, vertex_stage, pack_obs, half_rn, sincos, fk, collide, BACKGROUND_ID)  # noqa: F401
