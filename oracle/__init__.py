"""CPU oracle of the time-reversible FDTD gradient loop (arxiv/paper_2603_24027).

TEST INFRASTRUCTURE — NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import anything under oracle/.
"""
