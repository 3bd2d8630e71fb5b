"""CPU oracle of the Microcosmos step -- TEST INFRASTRUCTURE (see oracle/mco.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
may import this package.
"""
