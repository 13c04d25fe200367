"""Seeded synthetic inputs for the FlashNav simulator step.

This package holds INPUT DATA generators only (maps, robot specifications, action tapes, seeds).
It contains none of the method's arithmetic (no motion update, no ray casting, no collision test)
and is imported by the tests, by bench.py and by __graft_entry__.smoke(); neither `oracle/` nor
`paper_2606_15846_b200/` imports the other, and neither is imported from here.
"""
