"""CPU oracle of the FD Kohn-Sham apply -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import anything under oracle/.  Nothing here imports paper_2310_14776_b200.
"""
