"""Oracle: plain CPU implementation of the interval vote.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this package.  It never imports, and is never imported by, paper_2401_04576_b200's CUDA binding.
"""
