"""fp64 CPU oracle for libtabattn.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` leg may import anything under oracle/.  Nothing here
imports or is imported by paper_2606_03681_b200/.
"""
