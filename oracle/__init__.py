"""CPU oracle for the dipolar SSCN step — TEST INFRASTRUCTURE (see dbec_oracle.cpp header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import
this package.  It imports nothing from the product package.
"""
