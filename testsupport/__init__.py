"""Test-support code shared by tests/, bench.py and __graft_entry__.smoke():
the seeded synthetic input generators (SURVEY.md §8(d) "Synthetic inputs").  Nothing here is
part of the product package and nothing here does filter arithmetic; neither oracle/ nor
paper_1006_4644_b200/ imports it."""
