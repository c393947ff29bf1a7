"""Calibration microbenchmarks (not on the product path): the roofline denominators and the
structure limits quoted in DESIGN.md and profiles/.

    python -m paper_2505_03755_b200.calib            # builds with nvcc for sm_100a and runs on cuda:0
"""
