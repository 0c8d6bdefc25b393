"""oracle/ — TEST INFRASTRUCTURE, NOT THE PRODUCT.

A plain, slow, obviously-correct CPU statement of what the phx hot path computes,
written from /root/reference/PAPER.md and DESIGN.md's readings.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` leg may
import it.  It shares no code with paper_2607_01646_b200/ (neither imports the other).
"""
