"""CPU oracle for the ForeMoE plan + dispatch + combine path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2606_11867_b200.
"""
