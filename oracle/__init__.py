"""Float64 CPU oracle of the F-engine data path (arxiv 2303.09886).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It
shares no code with paper_2303_09886_b200 and never imports it.
"""
from .oracle import (  # noqa: F401
    build,
    lib,
    unpack10,
    unpack_bits,
    channelize_f64,
    process,
    direct_channel,
    fft_radix2,
    dft,
    fir,
    window,
    quantize,
    num_threads,
)
