from .processes import write_all

if __name__ == '__main__':
    for row in write_all():
        print(row)
